"""Thin Python binding over libnif.so (include/nif.h).  Same names as the C ABI.

Argument marshalling only: every step of the hot path runs in the CUDA kernels of libnif.so.
PyTorch is used for device memory and streams, nothing else.  There is no CPU fallback: if the
library is missing, or no sm_100 GPU is present, calls raise.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np
import torch

_HERE = Path(__file__).resolve().parent
LIB_PATH = _HERE / "libnif.so"

NIF_F32, NIF_F16 = 0, 1
NIF_ENC_COMPOSE, NIF_ENC_CONCAT = 0, 1
NIF_OCCLUSION_ONLY, NIF_ENGINE_FFMA, NIF_TRAVERSE_ONLY = 1, 2, 4
NIF_TRAVERSE_COHERENT, NIF_TRAVERSE_INCOHERENT, NIF_PROBE_SKIP_GATHER, NIF_DIST_LOG = 8, 16, 32, 64
NIF_N_OUT = 12
NIF_WALK_MISS, NIF_WALK_HIT, NIF_WALK_MAX_STEPS = 0, 1, 2


class NifError(RuntimeError):
    def __init__(self, status: int, what: str):
        self.status = status
        super().__init__(f"{what}: {lib().nif_error_string(status).decode()} ({status})")


class _VoxelSet(C.Structure):
    _fields_ = [("nv", C.c_int32), ("occupancy", C.c_void_p)]


class _DeformParams(C.Structure):
    _fields_ = [("twist_theta_max", C.c_float), ("bend_k", C.c_float)]


class _NetDesc(C.Structure):
    _fields_ = [("pe_bands", C.c_int32), ("levels", C.c_int32), ("log2_T", C.c_int32),
                ("feat", C.c_int32), ("level_res", C.POINTER(C.c_int32)),
                ("hidden_layers", C.c_int32), ("width", C.c_int32), ("dtype", C.c_int32),
                ("enc_mode", C.c_int32)]


class _RayBatch(C.Structure):
    _fields_ = [("n", C.c_int64), ("origin", C.c_void_p), ("dir", C.c_void_p)]


_OUT_FIELDS = ["voxel_id", "t_in", "t_out", "occlusion", "distance", "dist_total", "normal",
               "albedo", "material_logits", "raw_logits", "hit_position", "hit_position_rest"]


class _QueryOut(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in _OUT_FIELDS]


class _WalkOut(C.Structure):
    _fields_ = [("status", C.c_void_p), ("steps", C.c_void_p), ("dist_accum", C.c_void_p)]


class _BvhInfo(C.Structure):
    _fields_ = [("nv", C.c_int32), ("n_occupied", C.c_int32), ("n_nodes", C.c_int32),
                ("depth", C.c_int32), ("lo", C.c_float * 3), ("hi", C.c_float * 3),
                ("theta_max", C.c_float), ("bend_k", C.c_float)]


_lib = None


def lib() -> C.CDLL:
    """Loads libnif.so; fails loudly if it has not been built (no fallback path exists)."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise RuntimeError(f"{LIB_PATH} not built: run `python -m paper_2604_24666_b200.build` "
                               "(or __graft_entry__.build()); there is no CPU fallback")
        L = C.CDLL(str(LIB_PATH))
        L.nif_error_string.restype = C.c_char_p
        L.nif_error_string.argtypes = [C.c_int]
        L.nif_kernel_launch_count.restype = C.c_int64
        L.nif_bvh_workspace_bytes.argtypes = [C.c_int32, C.c_int64, C.POINTER(C.c_size_t)]
        L.nif_build_deformed_bvh.argtypes = [C.POINTER(_VoxelSet), C.POINTER(_DeformParams), C.c_void_p,
                                             C.c_size_t, C.c_void_p, C.POINTER(C.c_void_p)]
        L.nif_build_bvh_from_lattice.argtypes = [C.POINTER(_VoxelSet), C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p,
                                                 C.POINTER(C.c_void_p)]
        L.nif_bvh_refit_lattice.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.nif_bvh_refit.argtypes = [C.c_void_p, C.POINTER(_DeformParams), C.c_void_p]
        L.nif_bvh_get_info.argtypes = [C.c_void_p, C.POINTER(_BvhInfo)]
        L.nif_bvh_get_lattice.argtypes = [C.c_void_p, C.POINTER(C.c_void_p)]
        L.nif_bvh_destroy.argtypes = [C.c_void_p]
        L.nif_bvh_destroy.restype = None
        L.nif_net_create.argtypes = [C.POINTER(_NetDesc), C.c_void_p, C.POINTER(C.c_void_p), C.c_void_p,
                                     C.POINTER(C.c_void_p)]
        L.nif_net_destroy.argtypes = [C.c_void_p]
        L.nif_net_destroy.restype = None
        L.nif_net_uses_tensor_cores.argtypes = [C.c_void_p]
        L.nif_query_workspace_bytes.argtypes = [C.c_int64, C.POINTER(C.c_size_t)]
        L.nif_query.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(_RayBatch), C.POINTER(_QueryOut),
                                C.c_void_p, C.c_size_t, C.c_uint, C.c_void_p]
        L.nif_query_static.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(_RayBatch), C.POINTER(_QueryOut), C.c_uint, C.c_void_p]
        L.nif_query_poses_workspace_bytes.argtypes = [C.c_int64, C.POINTER(C.c_size_t)]
        L.nif_query_poses.argtypes = [C.POINTER(C.c_void_p), C.c_int32, C.c_void_p, C.POINTER(_RayBatch), C.c_void_p,
                                      C.POINTER(_QueryOut), C.c_void_p, C.c_size_t, C.c_uint, C.c_void_p]
        L.nif_query_multi_workspace_bytes.argtypes = [C.c_int64, C.POINTER(C.c_size_t)]
        L.nif_query_multi.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(_RayBatch), C.POINTER(_QueryOut),
                                      C.POINTER(_WalkOut), C.c_int32, C.c_void_p, C.c_size_t, C.c_uint, C.c_void_p]
        L.nif_stage_create.argtypes = [C.c_int64, C.POINTER(C.c_void_p)]
        L.nif_stage_destroy.argtypes = [C.c_void_p]
        L.nif_stage_destroy.restype = None
        L.nif_query_host.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(_RayBatch),
                                     C.POINTER(_QueryOut), C.c_uint]
        L.nif_query_last_hit_count.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_int64)]
        L.nif_profile_enable.argtypes = [C.c_int]
        L.nif_profile_read.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_int64)]
        L.nif_query_host_compact.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(_RayBatch), C.POINTER(_QueryOut),
                                             C.c_void_p, C.POINTER(C.c_int64), C.c_uint]
        L.nif_probe_gather.argtypes = [C.c_void_p, C.c_size_t, C.c_int, C.c_size_t, C.c_int, C.c_void_p,
                                       C.POINTER(C.c_double), C.POINTER(C.c_double)]
        _lib = L
    return _lib


def _check(status: int, what: str):
    if status != 0:
        raise NifError(status, what)


def _stream_ptr(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _ws(nbytes: int) -> torch.Tensor:
    t = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
    off = (-t.data_ptr()) % 256
    return t[off:off + nbytes]


def nif_kernel_launch_count() -> int:
    return int(lib().nif_kernel_launch_count())


def nif_bvh_workspace_bytes(nv: int, max_occupied: int) -> int:
    n = C.c_size_t()
    _check(lib().nif_bvh_workspace_bytes(nv, max_occupied, C.byref(n)), "nif_bvh_workspace_bytes")
    return n.value


class Bvh:
    """Owns the workspace tensor and the opaque nif_bvh handle."""

    def __init__(self, handle, workspace, occupancy):
        self.handle, self.workspace, self.occupancy = handle, workspace, occupancy

    def info(self) -> dict:
        i = _BvhInfo()
        _check(lib().nif_bvh_get_info(self.handle, C.byref(i)), "nif_bvh_get_info")
        return {"nv": i.nv, "n_occupied": i.n_occupied, "n_nodes": i.n_nodes, "depth": i.depth,
                "lo": np.array(list(i.lo), np.float32), "hi": np.array(list(i.hi), np.float32),
                "theta_max": i.theta_max, "bend_k": i.bend_k}

    def refit(self, theta_max: float, bend_k: float, stream=None):
        """nif_bvh_refit: new pose, same voxel set (synchronises)."""
        dp = _DeformParams(float(theta_max), float(bend_k))
        _check(lib().nif_bvh_refit(self.handle, C.byref(dp), _stream_ptr(stream)), "nif_bvh_refit")

    def refit_lattice(self, lattice_xyz: torch.Tensor, stream=None):
        """nif_bvh_refit_lattice: new user-specified deformed lattice [(nv+1)^3, 3] float32 CUDA (synchronises)."""
        assert lattice_xyz.is_cuda and lattice_xyz.dtype == torch.float32 and lattice_xyz.is_contiguous()
        _check(lib().nif_bvh_refit_lattice(self.handle, lattice_xyz.data_ptr(), _stream_ptr(stream)), "nif_bvh_refit_lattice")

    def lattice(self) -> torch.Tensor:
        """Copy of the deformed corner lattice, [(nv+1)^3, 3] float32 (for parity tests)."""
        p = C.c_void_p()
        _check(lib().nif_bvh_get_lattice(self.handle, C.byref(p)), "nif_bvh_get_lattice")
        nv = self.info()["nv"]
        n = (nv + 1) ** 3
        base = self.workspace.data_ptr()
        off = p.value - base
        flat = self.workspace[off:off + n * 16].view(torch.float32).view(n, 4)
        return flat[:, :3].clone()

    def __del__(self):
        try:
            if self.handle:
                lib().nif_bvh_destroy(self.handle)
                self.handle = None
        except Exception:
            pass


def nif_build_deformed_bvh(nv: int, occupancy: torch.Tensor, theta_max: float, bend_k: float,
                           max_occupied: int | None = None, stream=None) -> Bvh:
    """occupancy: uint8 CUDA tensor of nv^3 entries.  See include/nif.h."""
    assert occupancy.is_cuda and occupancy.dtype == torch.uint8 and occupancy.is_contiguous()
    assert occupancy.numel() == nv ** 3
    nbytes = nif_bvh_workspace_bytes(nv, nv ** 3 if max_occupied is None else max_occupied)
    ws = _ws(nbytes)
    vs = _VoxelSet(nv, occupancy.data_ptr())
    dp = _DeformParams(float(theta_max), float(bend_k))
    h = C.c_void_p()
    _check(lib().nif_build_deformed_bvh(C.byref(vs), C.byref(dp), ws.data_ptr(), nbytes,
                                        _stream_ptr(stream), C.byref(h)), "nif_build_deformed_bvh")
    return Bvh(h, ws, occupancy)


def nif_build_bvh_from_lattice(nv: int, occupancy: torch.Tensor, lattice_xyz: torch.Tensor,
                               max_occupied: int | None = None, stream=None) -> Bvh:
    """User-specified deformation given as the deformed corner lattice [(nv+1)^3, 3] float32 CUDA."""
    assert occupancy.is_cuda and occupancy.dtype == torch.uint8 and occupancy.is_contiguous()
    assert lattice_xyz.is_cuda and lattice_xyz.dtype == torch.float32 and lattice_xyz.is_contiguous()
    assert occupancy.numel() == nv ** 3 and lattice_xyz.numel() == 3 * (nv + 1) ** 3
    nbytes = nif_bvh_workspace_bytes(nv, nv ** 3 if max_occupied is None else max_occupied)
    ws = _ws(nbytes)
    vs = _VoxelSet(nv, occupancy.data_ptr())
    h = C.c_void_p()
    _check(lib().nif_build_bvh_from_lattice(C.byref(vs), lattice_xyz.data_ptr(), ws.data_ptr(), nbytes,
                                            _stream_ptr(stream), C.byref(h)), "nif_build_bvh_from_lattice")
    return Bvh(h, ws, occupancy)


class Net:
    def __init__(self, handle, keep):
        self.handle, self._keep = handle, keep

    def __del__(self):
        try:
            if self.handle:
                lib().nif_net_destroy(self.handle)
                self.handle = None
        except Exception:
            pass


def nif_net_create(shape, level_res, table: torch.Tensor, weights: list, stream=None) -> Net:
    """shape: object with pe_bands, levels, log2_T, feat, hidden_layers, width, dtype ("f32"|"f16").
    table: CUDA tensor [L, T, F]; weights: CUDA tensors (fan_out, fan_in); dtype per shape."""
    tdt = torch.float16 if shape.dtype == "f16" else torch.float32
    assert table.is_cuda and table.dtype == tdt and table.is_contiguous()
    for w in weights:
        assert w.is_cuda and w.dtype == tdt and w.is_contiguous()
    lr = np.ascontiguousarray(level_res, dtype=np.int32)
    d = _NetDesc(shape.pe_bands, shape.levels, shape.log2_T, shape.feat,
                 lr.ctypes.data_as(C.POINTER(C.c_int32)), shape.hidden_layers, shape.width,
                 NIF_F16 if shape.dtype == "f16" else NIF_F32,
                 NIF_ENC_CONCAT if getattr(shape, "enc_mode", "compose") == "concat" else NIF_ENC_COMPOSE)
    wp = (C.c_void_p * len(weights))(*[w.data_ptr() for w in weights])
    h = C.c_void_p()
    _check(lib().nif_net_create(C.byref(d), table.data_ptr(), wp, _stream_ptr(stream), C.byref(h)),
           "nif_net_create")
    return Net(h, (table, list(weights)))


def nif_net_uses_tensor_cores(net: Net) -> bool:
    r = lib().nif_net_uses_tensor_cores(net.handle)
    _check(min(r, 0), "nif_net_uses_tensor_cores")
    return bool(r)


def nif_query_workspace_bytes(n: int) -> int:
    b = C.c_size_t()
    _check(lib().nif_query_workspace_bytes(n, C.byref(b)), "nif_query_workspace_bytes")
    return b.value


def alloc_outputs(n: int, device="cuda", raw_logits: bool = False, pinned_host: bool = False,
                  hit_positions: bool = False) -> dict:
    kw = dict(device="cpu", pin_memory=True) if pinned_host else dict(device=device)
    o = {"voxel_id": torch.empty(n, dtype=torch.int32, **kw),
         "t_in": torch.empty(n, dtype=torch.float32, **kw),
         "t_out": torch.empty(n, dtype=torch.float32, **kw),
         "occlusion": torch.empty(n, dtype=torch.float32, **kw),
         "distance": torch.empty(n, dtype=torch.float32, **kw),
         "dist_total": torch.empty(n, dtype=torch.float32, **kw),
         "normal": torch.empty(n, 3, dtype=torch.float32, **kw),
         "albedo": torch.empty(n, 3, dtype=torch.float32, **kw),
         "material_logits": torch.empty(n, 4, dtype=torch.float32, **kw)}
    if raw_logits:
        o["raw_logits"] = torch.empty(n, NIF_N_OUT, dtype=torch.float32, **kw)
    if hit_positions:
        o["hit_position"] = torch.empty(n, 3, dtype=torch.float32, **kw)
        o["hit_position_rest"] = torch.empty(n, 3, dtype=torch.float32, **kw)
    return o


def _out_struct(out: dict) -> _QueryOut:
    q = _QueryOut()
    for k in _OUT_FIELDS:
        setattr(q, k, out[k].data_ptr() if k in out and out[k] is not None else None)
    return q


def nif_query(bvh: Bvh, net: Net | None, origin: torch.Tensor, direction: torch.Tensor, out: dict,
              workspace: torch.Tensor | None = None, flags: int = 0, stream=None) -> torch.Tensor:
    """Enqueues the query on the stream; returns the workspace tensor (reusable)."""
    n = origin.shape[0]
    assert origin.is_cuda and direction.is_cuda and origin.dtype == torch.float32
    assert origin.is_contiguous() and direction.is_contiguous() and direction.shape[0] == n
    if workspace is None:
        workspace = _ws(nif_query_workspace_bytes(n))
    rb = _RayBatch(n, origin.data_ptr(), direction.data_ptr())
    q = _out_struct(out)
    _check(lib().nif_query(bvh.handle, net.handle if net is not None else None, C.byref(rb), C.byref(q),
                           workspace.data_ptr(), workspace.numel(), flags, _stream_ptr(stream)), "nif_query")
    return workspace


NIF_STATIC_MAX_RAYS = 2097152          # include/nif.h


def nif_query_static(bvh: Bvh, net: Net | None, origin: torch.Tensor, direction: torch.Tensor, out: dict,
                     flags: int = 0, stream=None) -> None:
    """nif_query with the scratch in the library's own fixed device array: no allocation, at most
    NIF_STATIC_MAX_RAYS rays, calls that overlap on the GPU race (include/nif.h)."""
    n = origin.shape[0]
    assert origin.is_cuda and direction.is_cuda and origin.dtype == torch.float32
    assert origin.is_contiguous() and direction.is_contiguous() and direction.shape[0] == n
    rb = _RayBatch(n, origin.data_ptr(), direction.data_ptr())
    q = _out_struct(out)
    _check(lib().nif_query_static(bvh.handle, net.handle if net is not None else None, C.byref(rb), C.byref(q),
                                  flags, _stream_ptr(stream)), "nif_query_static")


def nif_query_poses_workspace_bytes(n: int) -> int:
    b = C.c_size_t()
    _check(lib().nif_query_poses_workspace_bytes(n, C.byref(b)), "nif_query_poses_workspace_bytes")
    return b.value


def nif_query_poses(bvhs: list, net: Net | None, origin: torch.Tensor, direction: torch.Tensor, pose_id: torch.Tensor,
                    out: dict, workspace: torch.Tensor | None = None, flags: int = 0, stream=None) -> torch.Tensor:
    """One query over rays of several poses: ray r is traced against bvhs[pose_id[r]] (include/nif.h)."""
    n = origin.shape[0]
    assert origin.is_cuda and direction.is_cuda and origin.dtype == torch.float32
    assert origin.is_contiguous() and direction.is_contiguous() and direction.shape[0] == n
    assert pose_id.is_cuda and pose_id.dtype == torch.int32 and pose_id.is_contiguous() and pose_id.numel() == n
    if workspace is None:
        workspace = _ws(nif_query_poses_workspace_bytes(n))
    rb = _RayBatch(n, origin.data_ptr(), direction.data_ptr())
    q = _out_struct(out)
    handles = (C.c_void_p * len(bvhs))(*[b.handle for b in bvhs])
    _check(lib().nif_query_poses(handles, len(bvhs), net.handle if net is not None else None, C.byref(rb),
                                 pose_id.data_ptr(), C.byref(q), workspace.data_ptr(), workspace.numel(), flags,
                                 _stream_ptr(stream)), "nif_query_poses")
    return workspace


def nif_query_multi_workspace_bytes(n: int) -> int:
    b = C.c_size_t()
    _check(lib().nif_query_multi_workspace_bytes(n, C.byref(b)), "nif_query_multi_workspace_bytes")
    return b.value


def alloc_walk_outputs(n: int, device="cuda") -> dict:
    return {"status": torch.empty(n, dtype=torch.int32, device=device),
            "steps": torch.empty(n, dtype=torch.int32, device=device),
            "dist_accum": torch.empty(n, dtype=torch.float32, device=device)}


def nif_query_multi(bvh: Bvh, net: Net, origin: torch.Tensor, direction: torch.Tensor, out: dict, walk: dict,
                    max_steps: int, workspace: torch.Tensor | None = None, flags: int = 0,
                    stream=None) -> torch.Tensor:
    """Multi-voxel walk (include/nif.h); enqueues on the stream, returns the workspace tensor."""
    n = origin.shape[0]
    assert origin.is_cuda and direction.is_cuda and origin.dtype == torch.float32
    assert origin.is_contiguous() and direction.is_contiguous() and direction.shape[0] == n
    if workspace is None:
        workspace = _ws(nif_query_multi_workspace_bytes(n))
    rb = _RayBatch(n, origin.data_ptr(), direction.data_ptr())
    q = _out_struct(out)
    w = _WalkOut(walk["status"].data_ptr(), walk["steps"].data_ptr(), walk["dist_accum"].data_ptr())
    _check(lib().nif_query_multi(bvh.handle, net.handle, C.byref(rb), C.byref(q), C.byref(w), int(max_steps),
                                 workspace.data_ptr(), workspace.numel(), flags, _stream_ptr(stream)),
           "nif_query_multi")
    return workspace


def nif_query_last_hit_count(workspace: torch.Tensor, stream=None) -> int:
    v = C.c_int64()
    _check(lib().nif_query_last_hit_count(workspace.data_ptr(), _stream_ptr(stream), C.byref(v)),
           "nif_query_last_hit_count")
    return v.value


def nif_profile_enable(on: bool):
    _check(lib().nif_profile_enable(1 if on else 0), "nif_profile_enable")


def nif_profile_read() -> dict:
    """Summed per-kernel milliseconds of the queries issued since the last read (synchronises)."""
    t, m, n = C.c_double(), C.c_double(), C.c_int64()
    _check(lib().nif_profile_read(C.byref(t), C.byref(m), C.byref(n)), "nif_profile_read")
    return {"traverse_ms": t.value, "network_ms": m.value, "n_queries": n.value}


def nif_probe_gather(buf: torch.Tensor, iters: int = 64, smem_bytes: int = 0, mode: int = 0, stream=None) -> dict:
    """Gather probe over `buf` (CUDA tensor): mode 0 = divergent lanes (L1 wavefront ceiling), mode 1 =
    warp-coalesced random lines (L2 / HBM sector rate); see include/nif.h."""
    assert buf.is_cuda and buf.is_contiguous()
    r, ms = C.c_double(), C.c_double()
    _check(lib().nif_probe_gather(buf.data_ptr(), buf.numel() * buf.element_size(), iters, smem_bytes, mode,
                                  _stream_ptr(stream), C.byref(r), C.byref(ms)), "nif_probe_gather")
    return {"sectors_per_s": r.value, "gbps": r.value * 32 / 1e9, "ms": ms.value}


def nif_query_host_compact(bvh: Bvh, net: Net | None, stage: "Stage", origin: torch.Tensor, direction: torch.Tensor,
                           out: dict, hit_ray: torch.Tensor, flags: int = 0) -> int:
    """nif_query_host with a compact return: dense voxel_id / t_in / t_out, head rows only for hit rays
    (row i belongs to ray hit_ray[i]).  All tensors HOST (ideally pinned).  Returns the number of hit rays."""
    n = origin.shape[0]
    assert not origin.is_cuda and not direction.is_cuda and origin.is_contiguous() and hit_ray.dtype == torch.int32
    rb = _RayBatch(n, origin.data_ptr(), direction.data_ptr())
    q = _out_struct(out)
    n_hit = C.c_int64()
    _check(lib().nif_query_host_compact(bvh.handle, net.handle if net is not None else None, stage.handle,
                                        C.byref(rb), C.byref(q), hit_ray.data_ptr(), C.byref(n_hit), flags),
           "nif_query_host_compact")
    return n_hit.value


class Stage:
    def __init__(self, chunk_rays: int):
        h = C.c_void_p()
        _check(lib().nif_stage_create(chunk_rays, C.byref(h)), "nif_stage_create")
        self.handle = h

    def __del__(self):
        try:
            if self.handle:
                lib().nif_stage_destroy(self.handle)
                self.handle = None
        except Exception:
            pass


def nif_query_host(bvh: Bvh, net: Net | None, stage: Stage, origin: torch.Tensor, direction: torch.Tensor,
                   out: dict, flags: int = 0):
    """origin/direction/out are HOST (ideally pinned) tensors; synchronises."""
    n = origin.shape[0]
    assert not origin.is_cuda and not direction.is_cuda and origin.is_contiguous()
    rb = _RayBatch(n, origin.data_ptr(), direction.data_ptr())
    q = _out_struct(out)
    _check(lib().nif_query_host(bvh.handle, net.handle if net is not None else None, stage.handle,
                                C.byref(rb), C.byref(q), flags), "nif_query_host")
