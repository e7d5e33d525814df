"""GPU-vs-oracle comparison used by the `-m gpu` parity tests.

Tolerances (BASELINE.json:5 north star; derivations in DESIGN.md section 8):
  voxel ids and hit/miss flags   bit-exact
  t_in, t_out                    |d| <= 1e-5 |ref|  (expected bit-equal; mismatches are counted)
  occlusion, albedo              max abs error <= 2e-2
  unit normal                    max abs error <= 2e-2 where the normalisation is well-conditioned (|z_n| >= 0.3 rms(z),
                                 >= 90 % of hit rays); everywhere: |dn| <= 2 |dz_n| / |z_n| (every normal error is
                                 explained by the gated logit error) and the decode arithmetic itself to 1e-5 (R29)
  distance                       s = sigmoid(z1): |d| <= tol; d: |d| <= tol*l + 1e-5 (t_in+t_out);
                                 D = t_in + d: relative <= tol;  tol = 1e-2 (fp16 MLP) / 1e-5 (fp32)
  material argmax                agreement >= 99.9 % of hit rays
  raw logits (sharper, ours)     max |dz| <= logit_tol * rms(z):  logit_tol = 5e-3 (fp16), 5e-5 (fp32)
"""
import numpy as np


def compare_traversal(gpu: dict, ref: dict) -> dict:
    gv = gpu["voxel_id"]; rv = ref["voxel_id"]
    assert gv.shape == rv.shape
    id_mismatch = int((gv != rv).sum())
    hit = rv >= 0
    both = hit & (gv >= 0)
    m = {"n": int(len(rv)), "n_hit": int(hit.sum()), "id_mismatch": id_mismatch}
    for k in ("t_in", "t_out"):
        g = gpu[k]; r = ref[k]
        m[k + "_bit_mismatch"] = int((g[both].view(np.int32) != r[both].view(np.int32)).sum())
        rel = np.abs(g[both] - r[both]) / np.maximum(np.abs(r[both]), 1e-30)
        m[k + "_max_rel"] = float(rel.max()) if rel.size else 0.0
        miss_ok = np.isinf(g[~hit]).all() and (g[~hit] > 0).all()
        m[k + "_miss_inf"] = bool(miss_ok)
    return m


def assert_traversal(m: dict):
    assert m["id_mismatch"] == 0, m
    assert m["t_in_max_rel"] <= 1e-5 and m["t_out_max_rel"] <= 1e-5, m
    assert m["t_in_miss_inf"] and m["t_out_miss_inf"], m


def compare_network(gpu: dict, ref: dict, fp16: bool, occlusion_only: bool = False) -> dict:
    hit = ref["voxel_id"] >= 0
    miss = ~hit
    m = {"n_hit": int(hit.sum())}
    keys = ["occlusion"] if occlusion_only else ["occlusion", "distance", "dist_total", "normal",
                                                  "albedo", "material_logits"]
    m["miss_all_zero"] = bool(all(not gpu[k][miss].any() for k in keys))
    m["occlusion_max_abs"] = float(np.abs(gpu["occlusion"][hit] - ref["occlusion"][hit]).max())
    if "raw_logits" in gpu and gpu["raw_logits"] is not None:
        cols = slice(0, 1) if occlusion_only else slice(0, 12)
        zr = ref["raw_logits"][hit][:, cols]; zg = gpu["raw_logits"][hit][:, cols]
        m["logit_rms"] = float(np.sqrt((zr.astype(np.float64) ** 2).mean()))
        m["logit_max_abs_over_rms"] = float(np.abs(zg - zr).max() / max(m["logit_rms"], 1e-30))
    if occlusion_only:
        return m
    tol = 1e-2 if fp16 else 1e-5
    m["tol"] = tol
    for k in ("albedo", "normal"):
        m[k + "_max_abs"] = float(np.abs(gpu[k][hit] - ref[k][hit]).max())
    if "raw_logits" in gpu and gpu["raw_logits"] is not None:
        # the unit normal z/|z| is ill-conditioned where the normal logits nearly vanish (random weights do
        # that, a trained head does not): |dn| <= 2 |dz| / |z|.  Views: the error where |z| >= 0.3 rms
        # (conditioned: the 2e-2 tolerance must hold), how many rays exceed 2e-2 at all, whether every
        # error is explained by the logit error (first-order bound), and the decode arithmetic itself
        # (GPU normal against the normalised GPU logits, fp64)
        zr = ref["raw_logits"][hit][:, 2:5].astype(np.float64); zg = gpu["raw_logits"][hit][:, 2:5].astype(np.float64)
        nr = np.linalg.norm(zr, axis=1); dz = np.linalg.norm(zg - zr, axis=1)
        dn = np.abs(gpu["normal"][hit] - ref["normal"][hit]).max(axis=1)
        cond = nr >= 0.3 * m["logit_rms"]
        m["normal_conditioned_frac"] = float(cond.mean())
        m["normal_conditioned_max_abs"] = float(dn[cond].max()) if cond.any() else 0.0
        m["normal_over_2e-2_count"] = int((dn > 2e-2).sum())
        m["normal_err_over_first_order_bound"] = float((dn / (2.0 * dz / np.maximum(nr, 1e-30) + 1e-6)).max())
        ng = zg / np.sqrt(np.maximum((zg * zg).sum(1, keepdims=True), 1e-24))
        m["normal_decode_max_abs"] = float(np.abs(gpu["normal"][hit] - ng).max())
    ti = ref["t_in"][hit].astype(np.float64); to = ref["t_out"][hit].astype(np.float64)
    ell = to - ti
    d_ref = ref["distance"][hit].astype(np.float64); d_gpu = gpu["distance"][hit].astype(np.float64)
    pos = ell > 0
    s_ref = np.where(pos, d_ref / np.where(pos, ell, 1), 0.0)
    ell_g = gpu["t_out"][hit].astype(np.float64) - gpu["t_in"][hit].astype(np.float64)
    s_gpu = np.where(ell_g > 0, d_gpu / np.where(ell_g > 0, ell_g, 1), 0.0)
    ok = pos & (ell_g > 0) & (ell > 1e-4)              # s is ill-defined on vanishing segments
    m["s_max_abs"] = float(np.abs(s_gpu[ok] - s_ref[ok]).max()) if ok.any() else 0.0
    bound = tol * ell + 1e-5 * (ti + to)
    m["distance_max_over_bound"] = float((np.abs(d_gpu - d_ref) / bound).max())
    D_ref = ref["dist_total"][hit].astype(np.float64); D_gpu = gpu["dist_total"][hit].astype(np.float64)
    m["dist_total_max_rel"] = float((np.abs(D_gpu - D_ref) / np.abs(D_ref)).max())
    am_ref = ref["material_logits"][hit].argmax(1); am_gpu = gpu["material_logits"][hit].argmax(1)
    m["material_argmax_agree"] = float((am_ref == am_gpu).mean())
    return m


def assert_network(m: dict, fp16: bool, occlusion_only: bool = False, logit_tol: float | None = None):
    assert m["miss_all_zero"], m
    assert m["occlusion_max_abs"] <= 2e-2, m
    if "logit_max_abs_over_rms" in m:
        assert m["logit_max_abs_over_rms"] <= (logit_tol or (5e-3 if fp16 else 5e-5)), m
    if occlusion_only:
        return
    assert m["albedo_max_abs"] <= 2e-2, m
    if "normal_conditioned_max_abs" in m:        # see compare_network; R29
        assert m["normal_conditioned_max_abs"] <= 2e-2 and m["normal_conditioned_frac"] >= 0.9, m
        assert m["normal_err_over_first_order_bound"] <= 1.0 and m["normal_decode_max_abs"] <= 1e-5, m
    else:
        assert m["normal_max_abs"] <= 2e-2, m
    assert m["s_max_abs"] <= m["tol"], m
    assert m["distance_max_over_bound"] <= 1.0, m
    assert m["dist_total_max_rel"] <= m["tol"], m
    assert m["material_argmax_agree"] >= 0.999, m
