"""TEST TOOLING: an independent numpy model of the shared-memory bank conflicts of backproject_scatter_kernel at the
paper-size geometry (cfg 4), used by tests/test_bank_model.py and quoted in DESIGN.md §5.

    python tests/bank_model.py            # the named layouts and a search over lane shapes, skews and pitches

A warp's 32 lanes scatter one trilinear sample each; an ATOMS.ADD instruction costs as many shared-memory wavefronts as
the largest number of lanes that fall on one of the 32 banks (atomics on the SAME word serialise too).  The eight corner
reductions of a sample are the same lane pattern shifted by a constant, so one bank histogram per sample suffices:
bank = (floor F + pS floor S + pZ floor Z) mod 32 with (F, S, Z) the sample position in (fast, slow, z) voxel indices.
Lanes are described by (pixel offset in u, pixel offset in v, sample-index skew).  "Merged" models the packed stream's
same-cell merging: the second sample of a pair only issues for lanes whose cell changed.
This restates geometry only; it shares nothing with the kernels or with tests/cpu_shim's own
bank statistics, which it reproduces (2.25 / 2.01 for the shipped layout) next to the one ncu figure there is (2.96 for
the 16 x 2 layout, profiles/README.md)."""
from __future__ import annotations

import numpy as np

NX = NY = 512; NZ = 70; DX = DY = 0.5; DZ = 2.5; NU = 512; NV = 384; DU = DV = 0.78; SAD = 1000.0; SDD = 1500.0; N_VIEWS = 40; STEP = 0.25
_R = float(np.sqrt((0.5 * (NX + 1) * DX) ** 2 + (0.5 * (NY + 1) * DY) ** 2 + (0.5 * (NZ + 1) * DZ) ** 2))
T_MIN, K = SAD - _R, int(np.ceil(2 * _R / STEP))


class Samples:
    """`trials` random (view, pixel tile, even sample index) positions, shared by every layout that is scored"""

    def __init__(self, trials=3000, seed=1):
        rng = np.random.default_rng(seed)
        self.theta = 2 * np.pi * rng.integers(0, N_VIEWS, trials) / N_VIEWS
        self.iu0, self.iv0 = rng.integers(0, NU - 64, trials), rng.integers(0, NV - 64, trials)
        self.k0 = 2 * rng.integers(100, (K - 300) // 2, trials)

    def floors(self, lu, lv, sk):
        c, s = np.cos(self.theta)[:, None], np.sin(self.theta)[:, None]
        u = (self.iu0[:, None] + lu[None, :] - (NU - 1) / 2) * DU
        v = (self.iv0[:, None] + lv[None, :] - (NV - 1) / 2) * DV
        ex, ey, ez = -SDD * c - u * s, -SDD * s + u * c, v
        L = np.sqrt(ex * ex + ey * ey + ez * ez)
        t = T_MIN + (self.k0[:, None] + sk[None, :] + 0.5) * STEP
        X, Y, Z = (SAD * c + ex / L * t) / DX + (NX - 1) / 2, (SAD * s + ey / L * t) / DY + (NY - 1) / 2, (ez / L * t) / DZ + (NZ - 1) / 2
        ok = ((X > -1) & (X < NX) & (Y > -1) & (Y < NY) & (Z > -1) & (Z < NZ)).all(axis=1)
        yfast = (np.abs(np.cos(self.theta)) > np.abs(np.sin(self.theta)))[:, None]      # the kernels' orientation rule
        F, S = np.where(yfast, Y, X), np.where(yfast, X, Y)
        return np.floor(F).astype(int), np.floor(S).astype(int), np.floor(Z).astype(int), ok


def _wavefronts(bank, active):
    hist = np.zeros((bank.shape[0], 32), int)
    rows = np.arange(bank.shape[0])[:, None].repeat(32, 1)
    np.add.at(hist, (rows[active], bank[active]), 1)
    return hist.max(axis=1)


def score(samples: Samples, lu, lv, sk, pS, pZ):
    """(wavefronts per ATOMS without merging, with same-cell merging, fraction of pairs in one cell)"""
    lu, lv, sk = np.asarray(lu), np.asarray(lv), np.asarray(sk)
    a, b = samples.floors(lu, lv, sk), samples.floors(lu, lv, sk + 1)
    ok = a[3] & b[3]
    bank_a, bank_b = (a[0] + pS * a[1] + pZ * a[2]) % 32, (b[0] + pS * b[1] + pZ * b[2]) % 32
    same = (a[0] == b[0]) & (a[1] == b[1]) & (a[2] == b[2])
    everyone = np.ones_like(same)
    w_a, w_b, w_b_all = _wavefronts(bank_a, everyone)[ok], _wavefronts(bank_b, ~same)[ok], _wavefronts(bank_b, everyone)[ok]
    return float((w_a.mean() + w_b_all.mean()) / 2), float((w_a.mean() + w_b.mean()) / 2), float(same[ok].mean())


LANES = np.arange(32)
LAYOUTS = {   # name: (du, dv, skew, row pitch mod 32, plane pitch mod 32)
    "LM1 16x2, rows 8 apart (ncu: 2.96)": (LANES & 15, (LANES >> 4) * 8, 0 * LANES, 8, 16),
    "LM0 8x4, two-sample skew per row (shipped)": (LANES & 7, LANES >> 3, 2 * (LANES >> 3), 8, 0),
    "8x4 without skew (ncu: 4.17)": (LANES & 7, LANES >> 3, 0 * LANES, 8, 16),
    "32x1, row pitch 0 mod 32": (LANES, 0 * LANES, 0 * LANES, 0, 0),
    "16x2, two-sample skew, row pitch 16 mod 32": (LANES & 15, LANES >> 4, 2 * (LANES >> 4), 16, 0),
}


def search(samples: Samples, widths=(8, 16, 32), skews=(0, 2, 4), plane_pitches=(0, 16)):
    """every lane shape W x (32/W), row skew and row / plane pitch mod 32: [(merged wavefronts per ATOMS, W, skew, pS, pZ)], best first"""
    out = []
    for W in widths:
        for sb in skews:
            lu, lv, sk = LANES % W, LANES // W, sb * (LANES // W)
            for pS in range(32):
                for pZ in plane_pitches:
                    out.append((score(samples, lu, lv, sk, pS, pZ)[1], W, sb, pS, pZ))
    return sorted(out)


if __name__ == "__main__":
    smp = Samples()
    for name, (lu, lv, sk, pS, pZ) in LAYOUTS.items():
        print("%-46s plain %.2f  merged %.2f  (pairs in one cell: %.0f %%)" % ((name,) + score(smp, lu, lv, sk, pS, pZ)[:2] + (100 * score(smp, lu, lv, sk, pS, pZ)[2],)))
    for r in search(smp)[:8]:
        print("search: %.3f  W=%d skew=%d row pitch %d plane pitch %d (mod 32)" % r)
