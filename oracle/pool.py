"""Runs the single-threaded CPU oracle over disjoint ray ranges on every core this process may use.

TEST INFRASTRUCTURE, part of the oracle package (same rule: only tests/, smoke() and bench.py's
cpu_baseline / --impl reference legs may import it): the `-m gpu` parity tests use it to put ALL rays of a
full-size configuration through the oracle ("Traversal parity runs on all rays of
every config"), and bench.py's cpu_baseline leg uses it for the all-cores figure.
The oracle function itself is unchanged and single-threaded; each worker process loads its own copy
of liboracle.so, builds its own oracle BVH from the lattice the parent computed once, and answers
chunks of rays.  Workers are spawned (not forked): the parent may hold a CUDA context.

Imports numpy, nif_inputs and oracle only -- never the CUDA package.
"""
from __future__ import annotations

import multiprocessing as mp
import os
import tempfile
from pathlib import Path

import numpy as np

_W = {}          # per-worker state


def n_cores() -> int:
    try:
        return max(1, len(os.sched_getaffinity(0)))
    except AttributeError:
        return max(1, os.cpu_count() or 1)


def cpu_model() -> str:
    try:
        for line in Path("/proc/cpuinfo").read_text().splitlines():
            if line.lower().startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def _init_worker(spec: dict) -> None:
    from oracle import Oracle
    import nif_inputs as I
    orc = Oracle()
    lat = np.load(spec["lattice_path"], mmap_mode="r")
    occ = np.ascontiguousarray(spec["occ"], dtype=np.uint8)
    bvh = orc.bvh_build(spec["nv"], occ, lat) if spec["build_bvh"] else None
    params = None
    if spec.get("table_path"):
        params = I.NetParams(spec["shape"], spec["level_res"], np.load(spec["table_path"], mmap_mode="r"),
                             spec["weights"], spec["variant"])
    _W.update(orc=orc, lat=lat, occ=occ, bvh=bvh, params=params, spec=spec)


def _run_chunk(args):
    o, d, kw = args
    s = _W["spec"]
    return _W["orc"].query(s["nv"], _W["occ"], _W["lat"], _W["bvh"], s["pose"], _W["params"], o, d, **kw)


class OraclePool:
    """Oracle side of one posed object (+ optionally one network) on `workers` processes."""

    def __init__(self, nv, occ, pose, lattice, params=None, workers: int | None = None, build_bvh: bool = True):
        self.workers = workers or n_cores()
        self._tmp = tempfile.TemporaryDirectory(prefix="nifo_pool_", dir="/dev/shm" if os.path.isdir("/dev/shm") else None)
        lat_path = os.path.join(self._tmp.name, "lattice.npy")
        np.save(lat_path, np.ascontiguousarray(lattice, dtype=np.float32))
        spec = {"nv": int(nv), "occ": np.ascontiguousarray(occ, dtype=np.uint8), "pose": [float(pose[0]), float(pose[1])],
                "lattice_path": lat_path, "build_bvh": build_bvh}
        if params is not None:
            tab_path = os.path.join(self._tmp.name, "table.npy")
            np.save(tab_path, np.ascontiguousarray(params.table, dtype=np.float32))
            spec.update(table_path=tab_path, shape=params.shape, level_res=params.level_res,
                        weights=params.weights, variant=params.variant)
        self._pool = mp.get_context("spawn").Pool(self.workers, initializer=_init_worker, initargs=(spec,))

    def query(self, origin, direction, chunk: int | None = None, **kw) -> dict:
        """oracle.query over all given rays; results concatenated in ray order."""
        n = len(origin)
        if n == 0:
            raise ValueError("empty batch")
        chunk = chunk or max(256, min(65536, -(-n // (self.workers * 8))))
        jobs = [(np.ascontiguousarray(origin[b:b + chunk]), np.ascontiguousarray(direction[b:b + chunk]), kw)
                for b in range(0, n, chunk)]
        parts = self._pool.map(_run_chunk, jobs, chunksize=1)
        return {k: np.concatenate([p[k] for p in parts]) for k in parts[0]}

    def close(self):
        if self._pool is not None:
            self._pool.close(); self._pool.join(); self._pool = None
            self._tmp.cleanup()

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            if self._pool is not None:
                self._pool.terminate(); self._tmp.cleanup()
        except Exception:
            pass
