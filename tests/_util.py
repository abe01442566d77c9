"""Shared helpers of the parity tests: the two error measures of BASELINE.json north_star
(reading F10 of DESIGN.md) and small wrappers that stream a workload through both sides."""
from __future__ import annotations

import numpy as np

REL_L2_TOL = 1e-5      # || z_gpu - z_ref ||_2 / || z_ref ||_2   per (stream, template), whole run
MAX_ABS_TOL = 1e-4     # max_k |z_gpu - z_ref| / max_k |z_ref|   per (stream, template), whole run


def parity_errors(z, ref):
    """z, ref: [..., n] complex; returns (worst rel-L2, worst max-abs ratio) over the leading axes."""
    z = np.asarray(z).reshape(ref.shape)
    num = np.sqrt((np.abs(z - ref) ** 2).sum(-1))
    den = np.sqrt((np.abs(ref) ** 2).sum(-1))
    mx = np.abs(z - ref).max(-1)
    mref = np.abs(ref).max(-1)
    ok = den > 0
    rel = np.where(ok, num / np.where(ok, den, 1.0), num)
    mab = np.where(mref > 0, mx / np.where(mref > 0, mref, 1.0), mx)
    return float(rel.max()), float(mab.max())


def assert_parity(z, ref, what=""):
    rel, mab = parity_errors(z, ref)
    assert rel <= REL_L2_TOL, f"{what}: rel-L2 {rel:.3e} > {REL_L2_TOL}"
    assert mab <= MAX_ABS_TOL, f"{what}: max-abs ratio {mab:.3e} > {MAX_ABS_TOL}"
    return rel, mab


def stream_gpu_plan(plan, blocks):
    """Run a list of float32 [S][n] numpy blocks through a paper_1702_02256_b200.Plan / MultiratePlan."""
    import torch
    outs = []
    for x in blocks:
        outs.append(plan.filter(torch.from_numpy(np.ascontiguousarray(x)).cuda()).cpu().numpy())
    torch.cuda.synchronize()
    return np.concatenate(outs, axis=-1)


def stream_oracle(orc, blocks):
    return np.concatenate([orc.filter(x) for x in blocks], axis=-1)


class ParityAccumulator:
    """The two error measures of F10 over a run that is compared block by block (full banks do not fit in
    host memory as one concatenated complex128 array): per (stream, template) sums of |dz|^2 and |z_ref|^2 and
    running maxima of |dz| and |z_ref| over the whole run."""

    def __init__(self):
        self.num = self.den = self.mx = self.mref = None

    def add(self, z, ref):
        z = np.asarray(z).reshape(ref.shape)
        d = np.abs(z - ref)
        r = np.abs(ref)
        num, den, mx, mref = (d ** 2).sum(-1), (r ** 2).sum(-1), d.max(-1), r.max(-1)
        if self.num is None:
            self.num, self.den, self.mx, self.mref = num, den, mx, mref
        else:
            self.num += num; self.den += den
            self.mx = np.maximum(self.mx, mx); self.mref = np.maximum(self.mref, mref)

    def check(self, what=""):
        rel = np.sqrt(self.num / np.where(self.den > 0, self.den, 1.0))
        mab = self.mx / np.where(self.mref > 0, self.mref, 1.0)
        assert np.all(self.den > 0), f"{what}: a reference series is identically zero"
        assert rel.max() <= REL_L2_TOL, f"{what}: rel-L2 {rel.max():.3e} > {REL_L2_TOL} (template {np.unravel_index(rel.argmax(), rel.shape)})"
        assert mab.max() <= MAX_ABS_TOL, f"{what}: max-abs ratio {mab.max():.3e} > {MAX_ABS_TOL}"
        return float(rel.max()), float(mab.max())
