"""CPU tests (-m "not gpu"): the C-ABI library loads and exports every symbol include/bs.h declares, the raw
JW term emitter agrees with the oracle's operator route (pin P3, second route), and the world-size-2 gloo
path of the row-slab sharding."""
import ctypes
import os
import re
import subprocess
import sys

import numpy as np
import pytest

import synth_inputs as si

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    from paper_2606_28952_b200 import build
    lib_path = build.build()
    hdr = open(os.path.join(ROOT, "include", "bs.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(bs_[a-z_0-9]+)\s*\(", hdr))
    assert {"bs_group_xmask", "bs_sector_build", "bs_apply", "bs_expect", "bs_apply_pauli_rotations"} <= declared
    lib = ctypes.CDLL(lib_path)
    for name in sorted(declared):
        assert hasattr(lib, name), f"libbs.so does not export {name}"
    from paper_2606_28952_b200 import bs
    assert set(bs.SYMBOLS) == declared
    lib.bs_version.restype = ctypes.c_char_p
    assert b"libbs" in lib.bs_version()
    lib.bs_launch_count.restype = ctypes.c_int64
    assert lib.bs_launch_count() == 0


def test_no_cpu_fallback_without_device():
    """Without a CUDA device every compute entry point fails loudly (BS_ERR_CUDA), never computes on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("needs a machine without a GPU")
    from paper_2606_28952_b200 import build
    lib = ctypes.CDLL(build.build())
    h = ctypes.c_void_p()
    rc = lib.bs_sector_build(6, 3, 3, None, ctypes.byref(h))
    assert rc == -3 and not h.value
    x = np.array([1], np.uint64)
    c = np.ones(1, np.complex128)
    rc = lib.bs_group_xmask(x.ctypes.data_as(ctypes.c_void_p), x.ctypes.data_as(ctypes.c_void_p),
                            c.ctypes.data_as(ctypes.c_void_p), ctypes.c_int64(1), 4, ctypes.c_double(0.0), 0, None,
                            ctypes.c_int64(0), None, ctypes.byref(h))
    assert rc == -3


def _merge(x, z, c, eps=1e-12):
    o = np.lexsort((z, x))
    x, z, c = x[o], z[o], c[o]
    head = np.ones(len(x), bool)
    head[1:] = (x[1:] != x[:-1]) | (z[1:] != z[:-1])
    cm = np.zeros(int(head.sum()), np.complex128)
    np.add.at(cm, np.cumsum(head) - 1, c)
    k = np.abs(cm) >= eps
    return x[head][k], z[head][k], cm[k]


@pytest.mark.parametrize("n", [2, 3, 6, 10])
def test_raw_terms_route_equals_oracle_route_molecular(n):
    from oracle import oracle as orc
    from paper_2606_28952_b200 import jw_terms as jw
    h, g = si.integrals(n, 500 + n)
    x, z, c = _merge(*jw.molecular_raw_terms(h, g))
    ref = orc.molecular_h(h, g)
    assert np.array_equal(x, ref.x) and np.array_equal(z, ref.z)
    assert np.abs(c - ref.c).max() <= 1e-13 * np.abs(ref.c).max()


def test_raw_terms_route_equals_oracle_route_hubbard_and_generators():
    from oracle import oracle as orc
    from paper_2606_28952_b200 import jw_terms as jw
    x, z, c = _merge(*jw.hubbard_raw_terms(14, 1.0, 4.0))
    ref = orc.hubbard_h(14, 1.0, 4.0)
    assert len(x) == 95 and np.array_equal(x, ref.x) and np.array_equal(z, ref.z) and np.abs(c - ref.c).max() == 0
    ex = si.uccsd_excitations(5, 2, 3)
    X, Z, C, offs = jw.excitation_generator_terms(ex)
    for j, (cre, ann) in enumerate(ex):
        o = orc.excitation_generator(cre, ann)
        s = slice(offs[j], offs[j + 1])
        assert np.array_equal(X[s], o.x) and np.array_equal(Z[s], o.z) and np.abs(C[s] - o.c).max() <= 1e-15
        assert np.all(np.abs(C[s].real) == 0) and len(o.x) in (2, 8)


def test_row_slabs():
    from paper_2606_28952_b200.dist import row_slabs
    for n, w in [(10, 3), (3432, 8), (5, 8), (0, 2), (20475, 7)]:
        s = row_slabs(n, w)
        assert len(s) == w and s[0][0] == 0 and s[-1][1] == n
        assert all(a[1] == b[0] for a, b in zip(s, s[1:]))
        lens = [b - a for a, b in s]
        assert max(lens) - min(lens) <= 1


WORKER = r"""
import os, sys
sys.path.insert(0, sys.argv[1])
import numpy as np, torch, torch.distributed as dist
import synth_inputs as si
from oracle import oracle as orc
from paper_2606_28952_b200.dist import sharded_apply, sharded_expect
dist.init_process_group("gloo")
rank = dist.get_rank()
for (n, na, nb) in [(6, 3, 3), (5, 2, 1)]:            # 20 rows (even slabs) and 10 rows of 5 (ragged for world 3, even for 2)
    h, g = si.integrals(n, 1001)
    ref = orc.molecular_h(h, g)
    osec = orc.Sector(n, na, nb)
    psi = si.random_state(osec.dim, 2001)
    def apply_rows(pin, pout, lo, hi):                # stand-in for bs_apply_rows: the oracle's slab apply
        out = np.full(osec.dim, np.nan + 0j)
        osec.apply_grouped(ref, pin.numpy(), lo, hi, out)
        pout[lo * osec.dim_beta:hi * osec.dim_beta] = torch.from_numpy(out[lo * osec.dim_beta:hi * osec.dim_beta])
    t_in = torch.from_numpy(psi.copy())
    t_out = torch.full_like(t_in, float('nan'))
    sharded_apply(apply_rows, t_in, t_out, osec.dim_alpha, osec.dim_beta)
    want = osec.apply(ref, psi)
    assert np.abs(t_out.numpy() - want).max() <= 1e-13, rank
    e = sharded_expect(apply_rows, t_in, torch.zeros_like(t_in), osec.dim_alpha, osec.dim_beta)
    assert abs(e - orc.vdot(psi, want)) <= 1e-12, rank
dist.barrier()
dist.destroy_process_group()
print("RANK_OK", rank)
"""


@pytest.mark.parametrize("world", [2, 3])
def test_sharded_apply_gloo(world, tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = 29600 + world + (os.getpid() % 200)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={world}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), str(script), ROOT]
    env = dict(os.environ, OMP_NUM_THREADS="1")
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, env=env)
    assert r.returncode == 0 and r.stdout.count("RANK_OK") == world, r.stdout[-2000:] + r.stderr[-3000:]


def test_bench_nonzero_count_matches_the_survey_table_and_the_oracle():
    """bench.py's flop count for the molecular configs (4 flops per non-zero) rests on the closed form for the
    non-zeros per row of H in a sector: 118 / 1,819 / 5,793 / 12,721 at configs 1, 2, 4, 5.
    At config 1 it is also counted by brute force from the oracle: the sector matrix of H, column by column."""
    import importlib.util
    from oracle import oracle as orc
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    spec = importlib.util.spec_from_file_location("bench_module", os.path.join(root, "bench.py"))
    bench = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(bench)
    want = {"q12": 118, "q24": 1819, "q32": 5793, "q56": 12721}
    for name, nnz in want.items():
        assert bench.nnz_per_row(si.CONFIGS[name]) == nnz
    cfg = si.CONFIGS["q12"]
    op = orc.molecular_h(*si.integrals(cfg.n_orb, cfg.seed_ints))
    sec = orc.Sector(cfg.n_orb, cfg.n_alpha, cfg.n_beta)
    eye = np.eye(sec.dim, dtype=np.complex128)
    # the grouped gather (one parallel region per call; pinned to the term-by-term definition by P12): the term-by-term
    # apply opens a parallel region per Pauli string, which takes minutes over 400 calls on a 400-dimensional sector
    hm = np.column_stack([sec.apply_grouped(op, eye[:, k].copy()) for k in range(sec.dim)])
    per_row = (np.abs(hm) > 1e-13).sum(axis=1)
    assert per_row.max() == 118 and int(per_row.sum()) == 47200      # generic integrals: every allowed element is non-zero
