"""Writes the full-size goldens of BASELINE.json configs[3] and configs[4] (32 and 56 qubits).

Calls ONLY the CPU oracle (oracle/) and the seeded input generators (synth_inputs.py); nothing from the CUDA
package is imported.  For the named config it evaluates H|psi> over the WHOLE sector with the oracle's Eq. 27
gather (orc_apply_grouped_slab, pinned to the term-by-term definition by P12) and stores

  energy          <psi|H|psi>              (Eq. 5), long-double accumulation over rows
  hnorm2          <H psi|H psi>
  row_e[D_a]      sum_j conj(psi[r, j]) (H psi)[r, j]   per alpha row r
  row_n2[D_a]     sum_j |(H psi)[r, j]|^2               per alpha row r
  sample_val[n]   (H psi)[t] for n seeded random targets t, by the DEFINITION (orc_apply_sampled: every Pauli
                  string visited for every target; SURVEY.md section 8(c) "sample of targets")

in tests/golden/fullsize_<config>.npz (+ the two scalars as text in tests/golden/energies.txt).  The GPU parity
test (tests/test_gpu_fullsize.py) compares bs_expect, the per-row functionals of bs_apply's output and the sampled
amplitudes with these values.  Rows are done in slabs and check-pointed, so an interrupted run resumes:

    OMP_NUM_THREADS=8 python tests/golden/make_fullsize_golden.py q32      # ~20 core-minutes... see README.md
    OMP_NUM_THREADS=8 python tests/golden/make_fullsize_golden.py q56      # hours on 8 cores
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
SAMPLE_SEED = 9


def sample_targets(dim: int) -> np.ndarray:
    return np.sort(np.random.default_rng(SAMPLE_SEED).integers(0, dim, N_SAMPLES)).astype(np.int64)


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("config", choices=["q24", "q32", "q56"])
    ap.add_argument("--slab", type=int, default=64, help="alpha rows per oracle call")
    ap.add_argument("--out", default=None)
    args = ap.parse_args()
    cfg = si.CONFIGS[args.config]
    out_path = args.out or os.path.join(HERE, f"fullsize_{cfg.name}.npz")
    ckpt = out_path + ".partial.npz"
    h, g = si.integrals(cfg.n_orb, cfg.seed_ints)
    op = orc.molecular_h(h, g)
    sec = orc.Sector(cfg.n_orb, cfg.n_alpha, cfg.n_beta)
    psi = si.random_state(cfg.dim, cfg.seed_psi)
    da, db = sec.dim_alpha, sec.dim_beta
    row_e = np.zeros(da, np.complex128)
    row_n2 = np.zeros(da, np.float64)
    done = 0
    if os.path.exists(ckpt):
        z = np.load(ckpt)
        done = int(z["done"])
        row_e[:done] = z["row_e"][:done]
        row_n2[:done] = z["row_n2"][:done]
        print(f"resuming at row {done}/{da}", flush=True)
    psi2 = psi.reshape(da, db)
    t0 = time.time()
    last = t0
    while done < da:
        hi = min(da, done + args.slab)
        out = sec.apply_grouped_slab(op, psi, done, hi)
        row_e[done:hi] = np.einsum("rj,rj->r", psi2[done:hi].conj(), out)
        row_n2[done:hi] = np.einsum("rj,rj->r", out.conj(), out).real
        done = hi
        if time.time() - last > 300 or done == da:
            np.savez(ckpt[:-4], done=done, row_e=row_e, row_n2=row_n2)
            last = time.time()
            print(f"rows {done}/{da}  {time.time() - t0:.0f} s", flush=True)
    energy = complex(np.sum(row_e.real.astype(np.longdouble)), np.sum(row_e.imag.astype(np.longdouble)))
    hnorm2 = float(np.sum(row_n2.astype(np.longdouble)))
    targets = sample_targets(cfg.dim)
    sample_val = sec.apply_sampled(op, psi, targets)
    np.savez_compressed(out_path[:-4], energy=np.array([energy.real, energy.imag]), hnorm2=hnorm2, row_e=row_e,
                        row_n2=row_n2, sample_seed=SAMPLE_SEED, sample_val=sample_val,
                        oracle_threads=orc.num_threads())
    # the two scalars as text
    txt = os.path.join(HERE, "energies.txt")
    lines = []
    if os.path.exists(txt):
        lines = [ln for ln in open(txt).read().splitlines() if ln and not ln.startswith(cfg.name + " ")]
    if not any(ln.startswith("#") for ln in lines):
        lines.insert(0, "# config  Re<psi|H|psi>  Im<psi|H|psi>  <Hpsi|Hpsi>   (written by make_fullsize_golden.py from oracle/ only)")
    lines.append(f"{cfg.name} {energy.real!r} {energy.imag!r} {hnorm2!r}")
    open(txt, "w").write("\n".join(lines) + "\n")
    if os.path.exists(ckpt):
        os.remove(ckpt)
    print(f"{cfg.name}: E = {energy.real!r} {energy.imag:+.3e}i  |H psi|^2 = {hnorm2!r}  ({time.time() - t0:.0f} s)")


if __name__ == "__main__":
    main()
