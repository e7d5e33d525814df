"""Sets one configuration up on both sides (CUDA path through the C ABI, CPU oracle) from the
same seeded inputs.  Used by the `-m gpu` tests only."""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np
import torch

import nif_inputs as I
import paper_2604_24666_b200 as nif


@dataclass
class Case:
    cfg: I.Config
    pose: np.ndarray
    occ: np.ndarray
    params: I.NetParams
    bvh: nif.Bvh
    net: nif.Net | None
    origin: np.ndarray
    direction: np.ndarray
    origin_d: torch.Tensor = None
    direction_d: torch.Tensor = None
    extra: dict = field(default_factory=dict)


def make_net(params: I.NetParams) -> nif.Net:
    table = torch.from_numpy(params.table_storage()).cuda()
    weights = [torch.from_numpy(w).cuda() for w in params.weights_storage()]
    return nif.nif_net_create(params.shape, params.level_res, table, weights)


def make_case(cfg_id: int, n_rays: int | None = None, variant: str = "varpres", pose_index: int = 0,
              with_net: bool = True, cfg: I.Config | None = None, occ=None, pose=None) -> Case:
    cfg = I.get_config(cfg_id) if cfg is None else cfg
    occ = I.occupancy(cfg) if occ is None else occ
    pose = I.poses(cfg)[pose_index] if pose is None else np.asarray(pose, np.float32)
    occ_d = torch.from_numpy(occ).cuda()
    bvh = nif.nif_build_deformed_bvh(cfg.nv, occ_d, float(pose[0]), float(pose[1]),
                                     max_occupied=int(occ.sum()))
    info = bvh.info()
    o, d = I.rays(cfg, pose_index, info["lo"], info["hi"], n=n_rays)
    params = I.net_params(cfg, variant)
    net = make_net(params) if with_net else None
    return Case(cfg, pose, occ, params, bvh, net, o, d,
                torch.from_numpy(o).cuda(), torch.from_numpy(d).cuda())


def run_gpu(case: Case, flags: int = 0, raw_logits: bool = True, hit_positions: bool = False) -> dict:
    n = len(case.origin)
    out = nif.alloc_outputs(n, raw_logits=raw_logits, hit_positions=hit_positions)
    for v in out.values():
        v.fill_(float("nan") if v.dtype.is_floating_point else -7)     # poison: everything must be written
    ws = nif.nif_query(case.bvh, case.net, case.origin_d, case.direction_d, out, flags=flags)
    torch.cuda.synchronize()
    res = {k: v.cpu().numpy() for k, v in out.items()}
    res["n_hit_counter"] = nif.nif_query_last_hit_count(ws)
    return res


class OracleSide:
    """Oracle lattice + BVH for a case (built once), queries on ray subsets."""

    def __init__(self, oracle, case: Case):
        self.oracle, self.case = oracle, case
        self.lattice = oracle.deform_lattice(case.cfg.nv, float(case.pose[0]), float(case.pose[1]))
        self.bvh = oracle.bvh_build(case.cfg.nv, case.occ, self.lattice)

    def query(self, idx=None, occlusion_only=False, traverse_only=False, **kw) -> dict:
        c = self.case
        o = c.origin if idx is None else c.origin[idx]
        d = c.direction if idx is None else c.direction[idx]
        return self.oracle.query(c.cfg.nv, c.occ, self.lattice, self.bvh, c.pose, c.params, o, d,
                                 occlusion_only=occlusion_only, traverse_only=traverse_only, **kw)


def subset(res: dict, idx) -> dict:
    return {k: (v[idx] if isinstance(v, np.ndarray) else v) for k, v in res.items()}
