"""Writes the full-list rotation golden of BASELINE.json configs[3] (32 qubits): tests/golden/fullsize_q32_rot.npz.

Calls ONLY the CPU oracle (oracle/) and the seeded input generators (synth_inputs.py); nothing from the CUDA package
is imported.  Step a6 (Eq. 39) on the config's seeded random state: all 5,792 first-order
Trotterised UCCSD generators of the (8, 8) sector of 16 orbitals, in the list order of reading U10
(synth_inputs.uccsd_excitations), angles synth_inputs.thetas(5792, 3004), each applied by the oracle's fermionic Givens
rotation (orc_rot_fermionic: SURVEY.md section 8(c) item 6, pinned by P9 against dense expm and against the product of
single-string Pauli rotations).  No Pauli strings are involved on this side.

Stored, so that the GPU test (tests/test_gpu_fullsize.py) can check the WHOLE rotated vector without holding a 2.65 GB
file:

  norm2            <psi'|psi'>, long-double accumulation
  row_sum[D_a]     sum_j psi'[r, j]      per alpha row r      (complex: sensitive to every phase in the row)
  row_n2[D_a]      sum_j |psi'[r, j]|^2  per alpha row r
  col_sum[D_b]     sum_r psi'[r, j]      per beta column j
  sample_idx[n], sample_val[n]   n = 65,536 seeded random amplitudes
  rows[4], row_val[4, D_b]       four complete alpha rows

    OMP_NUM_THREADS=8 python tests/golden/make_rotation_golden.py        # about half an hour on 8 cores
"""
from __future__ import annotations

import argparse
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

import synth_inputs as si  # noqa: E402
from oracle import oracle as orc  # noqa: E402

N_SAMPLES = 65536
SAMPLE_SEED = 11
THETA_SEED = 3004


def sample_targets(dim: int) -> np.ndarray:
    return np.sort(np.random.default_rng(SAMPLE_SEED).integers(0, dim, N_SAMPLES)).astype(np.int64)


def golden_rows(dim_alpha: int) -> np.ndarray:
    return np.array([0, dim_alpha // 3, (2 * dim_alpha) // 3, dim_alpha - 1], np.int64)


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", default="q32", choices=["q24", "q32"])
    ap.add_argument("--limit", type=int, default=None, help="only the first LIMIT generators (for a dry run)")
    ap.add_argument("--out", default=None)
    args = ap.parse_args()
    cfg = si.CONFIGS[args.config]
    out_path = args.out or os.path.join(HERE, f"fullsize_{cfg.name}_rot.npz")
    ex = si.uccsd_excitations(cfg.n_orb, cfg.n_alpha, cfg.n_beta)
    th = si.thetas(len(ex), THETA_SEED)
    n_gen = len(ex) if args.limit is None else min(args.limit, len(ex))
    sec = orc.Sector(cfg.n_orb, cfg.n_alpha, cfg.n_beta)
    da, db = sec.dim_alpha, sec.dim_beta
    psi = si.random_state(cfg.dim, cfg.seed_psi)
    t0 = time.time()
    for k in range(n_gen):
        cre, ann = ex[k]
        sec.rot_fermionic(psi, list(cre), list(ann), float(th[k]))
        if (k + 1) % 200 == 0 or k + 1 == n_gen:
            print(f"generator {k + 1}/{n_gen}  {time.time() - t0:.0f} s", flush=True)
    psi2 = psi.reshape(da, db)
    row_n2 = np.einsum("rj,rj->r", psi2.conj(), psi2).real
    norm2 = float(np.sum(row_n2.astype(np.longdouble)))
    targets = sample_targets(cfg.dim)
    rows = golden_rows(da)
    np.savez_compressed(out_path[:-4], n_generators=n_gen, theta_seed=THETA_SEED, norm2=norm2,
                        row_sum=psi2.sum(axis=1), row_n2=row_n2, col_sum=psi2.sum(axis=0),
                        sample_seed=SAMPLE_SEED, sample_idx=targets, sample_val=psi[targets],
                        rows=rows, row_val=psi2[rows], oracle_threads=orc.num_threads())
    print(f"{cfg.name}: {n_gen} generators, |psi'|^2 - 1 = {norm2 - 1.0:+.3e}  ({time.time() - t0:.0f} s) -> {out_path}")


if __name__ == "__main__":
    main()
