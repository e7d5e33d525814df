"""ctypes wrapper around oracle/nif_oracle.c -- the CPU oracle.

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It imports nothing from
paper_2604_24666_b200 and shares no code with it.  This file does argument marshalling only;
every formula lives in nif_oracle.c with its citation.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "nif_oracle.c"
_CFLAGS = ["-O2", "-std=c99", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC"]

FLAG_OCCLUSION_ONLY = 1
FLAG_DIST_LOG = 2
FLAG_LATTICE_INVERSE = 4
FLAG_ACT_F16 = 8
N_OUT = 12


def build(force: bool = False) -> dict:
    """Compile liboracle.so (acc float) and liboracle_acc64.so (acc double)."""
    out = {}
    for name, extra in (("liboracle.so", []), ("liboracle_acc64.so", ["-DNIFO_ACC_DOUBLE"])):
        so = _HERE / name
        if force or not so.exists() or so.stat().st_mtime < _SRC.stat().st_mtime:
            tmp = so.with_suffix(f".tmp{os.getpid()}.so")
            subprocess.check_call(["gcc", *_CFLAGS, *extra, str(_SRC), "-o", str(tmp), "-lquadmath", "-lm"])
            os.replace(tmp, so)
        out[name] = so
    return out


class _NetDesc(C.Structure):
    _fields_ = [("pe_bands", C.c_int32), ("levels", C.c_int32), ("log2_T", C.c_int32),
                ("feat", C.c_int32), ("hidden_layers", C.c_int32), ("width", C.c_int32),
                ("level_res", C.POINTER(C.c_int32)), ("enc_mode", C.c_int32)]


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _p(a, ty=C.c_float):
    return None if a is None else a.ctypes.data_as(C.POINTER(ty))


class Oracle:
    """One loaded oracle library.  acc64=True loads the double-accumulation build."""

    def __init__(self, acc64: bool = False):
        libs = build()
        self.lib = C.CDLL(str(libs["liboracle_acc64.so" if acc64 else "liboracle.so"]))
        L = self.lib
        L.nifo_bvh_build.restype = C.c_void_p
        L.nifo_bvh_build.argtypes = [C.c_int, C.c_void_p, C.c_void_p]
        L.nifo_bvh_destroy.argtypes = [C.c_void_p]
        L.nifo_bvh_num_voxels.argtypes = [C.c_void_p]
        L.nifo_bvh_bounds.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.nifo_traverse_bvh.argtypes = [C.c_void_p, C.c_int64] + [C.c_void_p] * 5
        L.nifo_traverse_brute.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_int64] + [C.c_void_p] * 5
        L.nifo_forward_f64.argtypes = [C.c_double, C.c_double, C.c_int64, C.c_void_p, C.c_void_p]
        L.nifo_deform_lattice.argtypes = [C.c_int, C.c_float, C.c_float, C.c_void_p]
        L.nifo_deform_lattice_counted.argtypes = [C.c_int, C.c_float, C.c_float, C.c_void_p, C.c_void_p]
        L.nifo_forward_exact_f32.argtypes = [C.c_float, C.c_float, C.c_int64, C.c_void_p, C.c_void_p]
        L.nifo_inverse_f32.argtypes = [C.c_float, C.c_float, C.c_int64, C.c_void_p, C.c_void_p]
        L.nifo_voxel_hit.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p,
                                     C.c_void_p, C.c_void_p]
        L.nifo_pe_samples.argtypes = [C.c_int, C.c_void_p, C.c_void_p]
        L.nifo_level_lookup.argtypes = [C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
        L.nifo_encode.argtypes = [C.POINTER(_NetDesc), C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
        L.nifo_mlp.argtypes = [C.POINTER(_NetDesc), C.c_void_p, C.c_int, C.c_int64, C.c_void_p, C.c_void_p]
        L.nifo_decode.argtypes = [C.c_int64] + [C.c_void_p] * 9
        L.nifo_round_f16.argtypes = [C.c_int64, C.c_void_p, C.c_void_p]
        L.nifo_query.restype = C.c_int
        L.nifo_query.argtypes = ([C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_float, C.c_float,
                                  C.POINTER(_NetDesc), C.c_void_p, C.c_void_p, C.c_int64,
                                  C.c_void_p, C.c_void_p, C.c_uint32] + [C.c_void_p] * 10)
        L.nifo_rest_endpoints.argtypes = [C.c_float, C.c_float, C.c_int64] + [C.c_void_p] * 6
        L.nifo_next_voxel_brute.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_int64] + [C.c_void_p] * 7
        L.nifo_next_voxel_bvh.argtypes = [C.c_void_p, C.c_int64] + [C.c_void_p] * 7
        L.nifo_query_multi.restype = C.c_int
        L.nifo_query_multi.argtypes = ([C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_float, C.c_float,
                                        C.POINTER(_NetDesc), C.c_void_p, C.c_void_p, C.c_int64,
                                        C.c_void_p, C.c_void_p, C.c_uint32, C.c_int] + [C.c_void_p] * 13)
        L.nifo_walk_trace.restype = C.c_int
        L.nifo_walk_trace.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_float, C.c_float,
                                      C.POINTER(_NetDesc), C.c_void_p, C.c_void_p, C.c_int64,
                                      C.c_void_p, C.c_void_p, C.c_uint32, C.c_int, C.c_void_p, C.c_void_p]
        L.nifo_hit_positions.argtypes = [C.c_void_p, C.c_int, C.c_uint32, C.c_float, C.c_float, C.c_int64] + [C.c_void_p] * 9
        L.nifo_inverse_trilinear.argtypes = [C.c_void_p, C.c_int, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p]
        L.nifo_exit_face_walk.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p,
                                          C.c_int, C.c_void_p, C.c_void_p]
        self.acc_bytes = L.nifo_acc_bytes()

    # ---- deformation -----------------------------------------------------------------
    def forward_f64(self, theta_max, k, p):
        p = np.ascontiguousarray(p, dtype=np.float64).reshape(-1, 3)
        out = np.empty_like(p)
        self.lib.nifo_forward_f64(float(theta_max), float(k), len(p), p.ctypes.data, out.ctypes.data)
        return out

    def deform_lattice(self, nv, theta_max, k, count_exact=False):
        """O2x: correctly rounded fp32 lattice (fp64 evaluation, binary128 where the rounding is in doubt)."""
        out = np.empty(((nv + 1) ** 3, 3), dtype=np.float32)
        cnt = C.c_int64(0)
        self.lib.nifo_deform_lattice_counted(int(nv), float(theta_max), float(k), out.ctypes.data, C.byref(cnt))
        return (out, cnt.value) if count_exact else out

    def forward_exact_f32(self, theta_max, k, p):
        """O2x definition: binary128 evaluation of the closed form, rounded once to fp32."""
        p = np.ascontiguousarray(p, dtype=np.float64).reshape(-1, 3)
        out = np.empty(p.shape, dtype=np.float32)
        self.lib.nifo_forward_exact_f32(float(theta_max), float(k), len(p), p.ctypes.data, out.ctypes.data)
        return out

    def inverse_trilinear(self, lattice, nv, voxel_id, P):
        """O7b: rest points of P[i], each taken to lie in deformed voxel voxel_id[i]."""
        P = _f32(P).reshape(-1, 3)
        vid = np.ascontiguousarray(voxel_id, dtype=np.int32)
        out = np.empty_like(P)
        self.lib.nifo_inverse_trilinear(lattice.ctypes.data, int(nv), len(P), vid.ctypes.data, P.ctypes.data, out.ctypes.data)
        return out

    def inverse_f32(self, theta_max, k, P):
        P = _f32(P).reshape(-1, 3)
        out = np.empty_like(P)
        self.lib.nifo_inverse_f32(float(theta_max), float(k), len(P), P.ctypes.data, out.ctypes.data)
        return out

    # ---- traversal -------------------------------------------------------------------
    def voxel_hit(self, lattice, nv, voxel_id, o, d):
        o = _f32(o); d = _f32(d)
        ti = C.c_float(); to = C.c_float()
        hit = self.lib.nifo_voxel_hit(lattice.ctypes.data, nv, int(voxel_id), o.ctypes.data,
                                      d.ctypes.data, C.byref(ti), C.byref(to))
        return bool(hit), ti.value, to.value

    def traverse_brute(self, nv, occ, lattice, origin, direction):
        origin = _f32(origin); direction = _f32(direction)
        n = len(origin)
        vid = np.empty(n, np.int32); ti = np.empty(n, np.float32); to = np.empty(n, np.float32)
        self.lib.nifo_traverse_brute(nv, occ.ctypes.data, lattice.ctypes.data, n, origin.ctypes.data,
                                     direction.ctypes.data, vid.ctypes.data, ti.ctypes.data, to.ctypes.data)
        return vid, ti, to

    def bvh_build(self, nv, occ, lattice):
        return OracleBVH(self, nv, occ, lattice)

    # ---- encoding / network ----------------------------------------------------------
    def _desc(self, shape, level_res):
        lr = np.ascontiguousarray(level_res, dtype=np.int32)
        d = _NetDesc(shape.pe_bands, shape.levels, shape.log2_T, shape.feat,
                     shape.hidden_layers, shape.width, lr.ctypes.data_as(C.POINTER(C.c_int32)),
                     1 if getattr(shape, "enc_mode", "compose") == "concat" else 0)
        d._keep = lr
        return d

    def pe_samples(self, bands, xn):
        xn = _f32(xn)
        out = np.empty((1 + 2 * bands, 3), np.float32)
        self.lib.nifo_pe_samples(bands, xn.ctypes.data, out.ctypes.data)
        return out

    def level_lookup(self, N, log2_T, p):
        p = _f32(p)
        idx = np.empty(8, np.uint32); w = np.empty(8, np.float32)
        self.lib.nifo_level_lookup(int(N), int(log2_T), p.ctypes.data, idx.ctypes.data, w.ctypes.data)
        return idx, w

    def encode(self, params, xn):
        """psi(x_n) for n normalised points -> [n, S*L*F]"""
        sh = params.shape
        xn = _f32(xn).reshape(-1, 3)
        d = self._desc(sh, params.level_res)
        table = _f32(params.table)
        out = np.empty((len(xn), sh.d_in // 2), np.float32)
        self.lib.nifo_encode(C.byref(d), table.ctypes.data, len(xn), xn.ctypes.data, out.ctypes.data)
        return out

    def _wptrs(self, weights):
        ws = [_f32(w) for w in weights]
        arr = (C.c_void_p * len(ws))(*[w.ctypes.data for w in ws])
        return ws, arr

    def mlp(self, params, x):
        sh = params.shape
        x = _f32(x)
        d = self._desc(sh, params.level_res)
        ws, arr = self._wptrs(params.weights)
        out = np.empty((len(x), N_OUT), np.float32)
        self.lib.nifo_mlp(C.byref(d), arr, x.shape[1], len(x), x.ctypes.data, out.ctypes.data)
        return out

    def round_f16(self, x):
        """O9b: IEEE binary16 round-to-nearest-even of each value, as float32"""
        x = _f32(x)
        out = np.empty_like(x)
        self.lib.nifo_round_f16(x.size, x.ctypes.data, out.ctypes.data)
        return out

    def decode(self, logits, t_in, t_out):
        logits = _f32(logits); t_in = _f32(t_in); t_out = _f32(t_out)
        n = len(logits)
        o = {"occlusion": np.empty(n, np.float32), "distance": np.empty(n, np.float32),
             "dist_total": np.empty(n, np.float32), "normal": np.empty((n, 3), np.float32),
             "albedo": np.empty((n, 3), np.float32), "material_logits": np.empty((n, 4), np.float32)}
        self.lib.nifo_decode(n, logits.ctypes.data, t_in.ctypes.data, t_out.ctypes.data,
                             o["occlusion"].ctypes.data, o["distance"].ctypes.data,
                             o["dist_total"].ctypes.data, o["normal"].ctypes.data,
                             o["albedo"].ctypes.data, o["material_logits"].ctypes.data)
        return o

    def rest_endpoints(self, theta_max, k, origin, direction, vid, t_in, t_out):
        origin = _f32(origin); direction = _f32(direction)
        out = np.empty((len(origin), 2, 3), np.float32)
        self.lib.nifo_rest_endpoints(float(theta_max), float(k), len(origin), origin.ctypes.data,
                                     direction.ctypes.data, vid.ctypes.data, t_in.ctypes.data,
                                     t_out.ctypes.data, out.ctypes.data)
        return out

    def query(self, nv, occ, lattice, bvh, pose, params, origin, direction,
              occlusion_only=False, traverse_only=False, dist_log=False, hit_positions=False,
              lattice_inverse=False, act_f16=False):
        """Whole pipeline.  bvh=None -> brute-force definition.  act_f16: O9b (fp16 activations, B:8)."""
        origin = _f32(origin); direction = _f32(direction)
        n = len(origin)
        sh = params.shape
        d = self._desc(sh, params.level_res)
        table = _f32(params.table)
        ws, arr = self._wptrs(params.weights)
        o = {"voxel_id": np.empty(n, np.int32), "t_in": np.empty(n, np.float32),
             "t_out": np.empty(n, np.float32)}
        if not traverse_only:
            o.update({"occlusion": np.zeros(n, np.float32), "distance": np.zeros(n, np.float32),
                      "dist_total": np.zeros(n, np.float32), "normal": np.zeros((n, 3), np.float32),
                      "albedo": np.zeros((n, 3), np.float32),
                      "material_logits": np.zeros((n, 4), np.float32),
                      "raw_logits": np.zeros((n, N_OUT), np.float32)})
        g = lambda k: (o[k].ctypes.data if k in o else None)
        rc = self.lib.nifo_query(nv, occ.ctypes.data, lattice.ctypes.data,
                                 bvh.handle if bvh is not None else None,
                                 float(pose[0]), float(pose[1]), C.byref(d), table.ctypes.data, arr,
                                 n, origin.ctypes.data, direction.ctypes.data,
                                 (FLAG_OCCLUSION_ONLY if occlusion_only else 0) | (FLAG_DIST_LOG if dist_log else 0) |
                                 (FLAG_LATTICE_INVERSE if lattice_inverse else 0) | (FLAG_ACT_F16 if act_f16 else 0),
                                 g("voxel_id"), g("t_in"), g("t_out"), g("occlusion"), g("distance"),
                                 g("dist_total"), g("normal"), g("albedo"), g("material_logits"),
                                 g("raw_logits"))
        if rc != 0:
            raise RuntimeError(f"nifo_query failed: {rc}")
        if hit_positions and not traverse_only and not occlusion_only:
            o["hit_position"], o["hit_position_rest"] = self.hit_positions(
                pose, origin, direction, o, lattice=lattice if lattice_inverse else None, nv=nv)
        return o

    def hit_positions(self, pose, origin, direction, res, lattice=None, nv=0):
        """O12: (deformed-space, rest-space) hit positions from a query's outputs (lattice given: O7b inverse)."""
        origin = _f32(origin); direction = _f32(direction)
        n = len(origin)
        hp = np.empty((n, 3), np.float32); hr = np.empty((n, 3), np.float32)
        self.lib.nifo_hit_positions(lattice.ctypes.data if lattice is not None else None, int(nv),
                                    FLAG_LATTICE_INVERSE if lattice is not None else 0,
                                    float(pose[0]), float(pose[1]), n, origin.ctypes.data, direction.ctypes.data,
                                    res["voxel_id"].ctypes.data, res["t_in"].ctypes.data, res["t_out"].ctypes.data,
                                    res["distance"].ctypes.data, res["dist_total"].ctypes.data,
                                    hp.ctypes.data, hr.ctypes.data)
        return hp, hr


    def exit_face_walk(self, nv, occ, lattice, bvh, origin, direction, max_vox):
        """O11x: the literal exit-face walk of P:51 -> (seq [n, max_vox] of occupied voxel ids, -1 padded; status [n])."""
        origin = _f32(origin); direction = _f32(direction)
        n = len(origin)
        seq = np.empty((n, max_vox), np.int32); status = np.empty(n, np.int32)
        self.lib.nifo_exit_face_walk(int(nv), occ.ctypes.data, lattice.ctypes.data, bvh.handle if bvh is not None else None,
                                     n, origin.ctypes.data, direction.ctypes.data, int(max_vox), seq.ctypes.data, status.ctypes.data)
        return seq, status

    def next_voxel_brute(self, nv, occ, lattice, origin, direction, after_t, after_id):
        """O11 definition: successor of (after_t, after_id) in each ray's (t_in, id)-ordered voxel sequence."""
        origin = _f32(origin); direction = _f32(direction)
        at = _f32(after_t); ai = np.ascontiguousarray(after_id, dtype=np.int32)
        n = len(origin)
        vid = np.empty(n, np.int32); ti = np.empty(n, np.float32); to = np.empty(n, np.float32)
        self.lib.nifo_next_voxel_brute(nv, occ.ctypes.data, lattice.ctypes.data, n, origin.ctypes.data,
                                       direction.ctypes.data, at.ctypes.data, ai.ctypes.data,
                                       vid.ctypes.data, ti.ctypes.data, to.ctypes.data)
        return vid, ti, to

    def query_multi(self, nv, occ, lattice, bvh, pose, params, origin, direction, max_steps,
                    occlusion_only=False, lattice_inverse=False):
        """O11: multi-voxel walk; returns the single-voxel outputs of the accepted (or last) voxel plus
        status / steps / dist_accum (the literal P:61 sum)."""
        origin = _f32(origin); direction = _f32(direction)
        n = len(origin)
        d = self._desc(params.shape, params.level_res)
        table = _f32(params.table)
        ws, arr = self._wptrs(params.weights)
        o = {"voxel_id": np.empty(n, np.int32), "t_in": np.empty(n, np.float32), "t_out": np.empty(n, np.float32),
             "occlusion": np.zeros(n, np.float32), "distance": np.zeros(n, np.float32),
             "dist_total": np.zeros(n, np.float32), "normal": np.zeros((n, 3), np.float32),
             "albedo": np.zeros((n, 3), np.float32), "material_logits": np.zeros((n, 4), np.float32),
             "raw_logits": np.zeros((n, N_OUT), np.float32), "status": np.zeros(n, np.int32),
             "steps": np.zeros(n, np.int32), "dist_accum": np.zeros(n, np.float32)}
        rc = self.lib.nifo_query_multi(nv, occ.ctypes.data, lattice.ctypes.data,
                                       bvh.handle if bvh is not None else None,
                                       float(pose[0]), float(pose[1]), C.byref(d), table.ctypes.data, arr,
                                       n, origin.ctypes.data, direction.ctypes.data,
                                       (FLAG_OCCLUSION_ONLY if occlusion_only else 0) |
                                       (FLAG_LATTICE_INVERSE if lattice_inverse else 0), int(max_steps),
                                       *[o[k].ctypes.data for k in ("voxel_id", "t_in", "t_out", "occlusion",
                                                                    "distance", "dist_total", "normal", "albedo",
                                                                    "material_logits", "raw_logits", "status",
                                                                    "steps", "dist_accum")])
        if rc != 0:
            raise RuntimeError(f"nifo_query_multi failed: {rc}")
        return o


    def walk_trace(self, nv, occ, lattice, bvh, pose, params, origin, direction, max_steps, lattice_inverse=False):
        """O11 trace: (trace_id, trace_z0), each [n, max_steps]; id -1 past the end of a ray's voxel sequence."""
        origin = _f32(origin); direction = _f32(direction)
        n = len(origin)
        d = self._desc(params.shape, params.level_res)
        table = _f32(params.table)
        ws, arr = self._wptrs(params.weights)
        tid = np.empty((n, max_steps), np.int32); tz = np.empty((n, max_steps), np.float32)
        rc = self.lib.nifo_walk_trace(nv, occ.ctypes.data, lattice.ctypes.data,
                                      bvh.handle if bvh is not None else None, float(pose[0]), float(pose[1]),
                                      C.byref(d), table.ctypes.data, arr, n, origin.ctypes.data,
                                      direction.ctypes.data, FLAG_LATTICE_INVERSE if lattice_inverse else 0,
                                      int(max_steps), tid.ctypes.data, tz.ctypes.data)
        if rc != 0:
            raise RuntimeError(f"nifo_walk_trace failed: {rc}")
        return tid, tz


class OracleBVH:
    def __init__(self, oracle: Oracle, nv, occ, lattice):
        self.oracle = oracle
        self.nv = nv
        self.occ = np.ascontiguousarray(occ, dtype=np.uint8)
        self.lattice = _f32(lattice)               # borrowed by the C side: keep alive
        self.handle = oracle.lib.nifo_bvh_build(nv, self.occ.ctypes.data, self.lattice.ctypes.data)

    def bounds(self):
        lo = np.empty(3, np.float32); hi = np.empty(3, np.float32)
        self.oracle.lib.nifo_bvh_bounds(self.handle, lo.ctypes.data, hi.ctypes.data)
        return lo, hi

    def num_voxels(self):
        return self.oracle.lib.nifo_bvh_num_voxels(self.handle)

    def traverse(self, origin, direction):
        origin = _f32(origin); direction = _f32(direction)
        n = len(origin)
        vid = np.empty(n, np.int32); ti = np.empty(n, np.float32); to = np.empty(n, np.float32)
        self.oracle.lib.nifo_traverse_bvh(self.handle, n, origin.ctypes.data, direction.ctypes.data,
                                          vid.ctypes.data, ti.ctypes.data, to.ctypes.data)
        return vid, ti, to

    def next_voxel(self, origin, direction, after_t, after_id):
        origin = _f32(origin); direction = _f32(direction)
        at = _f32(after_t); ai = np.ascontiguousarray(after_id, dtype=np.int32)
        n = len(origin)
        vid = np.empty(n, np.int32); ti = np.empty(n, np.float32); to = np.empty(n, np.float32)
        self.oracle.lib.nifo_next_voxel_bvh(self.handle, n, origin.ctypes.data, direction.ctypes.data,
                                            at.ctypes.data, ai.ctypes.data, vid.ctypes.data, ti.ctypes.data,
                                            to.ctypes.data)
        return vid, ti, to

    def __del__(self):
        try:
            self.oracle.lib.nifo_bvh_destroy(self.handle)
        except Exception:
            pass
