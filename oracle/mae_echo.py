"""RoPE-logit MAE on synthetic data: the direction check of the paper's Table 1.

Calls only oracle/ and the seeded input generators (workloads/).  `python -m oracle.mae_echo` prints the table quoted in
BASELINE.md: uniform TQ-MSE vs Block-GTQ (greedy allocation from the block-energy scores of a SEPARATE calibration draw),
each with the shared Gaussian codebooks (reading Q7) and with the exact-density (sphere-marginal) codebooks, at 2 and
3 bits per dimension, on Qwen2.5-3B-shaped heads (16 query / 2 KV heads, d_h = 128, theta base 1e6) whose RoPE blocks have
log-uniform energies over three decades (DESIGN.md section 5 -- stands in for WikiText-2 activations, which are not here).
"""
from __future__ import annotations

import sys

import numpy as np

import workloads as W
from oracle import oracle as O


def table(n_eval: int = 256, n_cal: int = 512, seeds=(2, 3, 4), budgets=(2, 3), d: int = 128, Hq: int = 16, Hkv: int = 2,
          base: float = 1.0e6, rot_seed: int = 20260624):
    rot = W.rotations(rot_seed, d)
    tabs = {"gaussian": O.Tables(rot, d), "sphere": O.Tables(rot, d, cb_kind="sphere")}
    rows = []
    for bbar in budgets:
        acc = {(m, c): [] for m in ("uniform", "block-gtq") for c in tabs}
        for seed in seeds:
            scales = W.block_scales(seed, Hkv, d // 2)
            q_cal = W.pre_rope_gaussian(seed, 4, n_cal, Hq, d, scales)
            k_cal = W.pre_rope_gaussian(seed, 1, n_cal, Hkv, d, scales)
            s, _, _ = O.block_energy(q_cal, k_cal)
            greedy = np.stack([O.allocate(s[h], bbar * (d // 2), 1, 8) for h in range(Hkv)])
            uniform = np.full_like(greedy, bbar)
            q = W.pre_rope_gaussian(seed, 5, n_eval, Hq, d, scales)
            k = W.pre_rope_gaussian(seed, 6, n_eval, Hkv, d, scales)
            for cname, tab in tabs.items():
                acc[("uniform", cname)].append(O.rope_logit_mae(q, k, uniform, tab, base))
                acc[("block-gtq", cname)].append(O.rope_logit_mae(q, k, greedy, tab, base))
        rows.append((bbar, {k: float(np.mean(v)) for k, v in acc.items()}))
    return rows


if __name__ == "__main__":
    n = int(sys.argv[1]) if len(sys.argv) > 1 else 256
    print("| budget | uniform TQ-MSE (Gaussian C_b) | Block-GTQ (Gaussian C_b) | reduction | uniform (exact-density C_b,m) | Block-GTQ (exact-density C_b,m) | reduction |")
    print("|---|---|---|---|---|---|---|")
    for bbar, r in table(n_eval=n):
        ug, bg, us, bs = r[("uniform", "gaussian")], r[("block-gtq", "gaussian")], r[("uniform", "sphere")], r[("block-gtq", "sphere")]
        print(f"| {bbar} b/dim | {ug:.4f} | {bg:.4f} | {100 * (1 - bg / ug):+.1f} % | {us:.4f} | {bs:.4f} | {100 * (1 - bs / us):+.1f} % |")
