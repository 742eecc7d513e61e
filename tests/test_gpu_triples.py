"""GPU parity of the perturbative triples (Appendix 7.3) against the triples oracle.

Per-term: the dense blocks Wbar, Zbar, Ybar [a][b][c] of sampled occupied triples, element by element (1e-12 relative
max-abs).  Energies: E(+T), E((T)), E(-T) (Re and Im) within 1e-10 Eh at seeded random amplitudes and at the oracle's
CCSD iterate.  Shapes: cfg0, a ragged one (several DMMA tiles with tails in every dimension, odd nvir -> the kernel
variant without sum planes), cfg1 (sampled blocks live, energies against tests/golden/oracle_triples_cfg1.txt).
"""
import os

import numpy as np
import pytest

import ccsd_inputs as ci

pytestmark = pytest.mark.gpu

REL_TOL = 1e-12
E_TOL = 1e-10
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2103_08473_b200 as lib
    lib.load_library()
    return lib


def _rel(a, b):
    scale = np.abs(b).max()
    return np.abs(np.asarray(a) - np.asarray(b)).max() / (scale if scale > 0 else 1.0)


def _pair(cfg):
    from oracle.ccsd_oracle import OracleCCSD
    if cfg == "ragged":
        inp = ci.make_inputs(7, 29, 37, seed=4711)
    elif cfg == "ragged_even":
        inp = ci.make_inputs(5, 38, 30, seed=4712)
    else:
        inp = ci.make_config(cfg)
    oc = OracleCCSD(inp.h, inp.B, inp.nocc, inp.nvir, restricted=inp.nvir > 40)
    return inp, oc


@pytest.mark.parametrize("cfg,scale,triples", [
    ("cfg0", 0.2, [(0, 1, 2), (0, 1, 3), (1, 2, 3)]),
    ("ragged", 0.05, [(0, 1, 2), (1, 3, 6), (4, 5, 6)]),
    ("ragged_even", 0.05, [(0, 2, 4), (2, 3, 4)]),
    ("cfg1", 0.01, [(0, 1, 2), (3, 9, 15), (13, 14, 15)]),
])
def test_triples_blocks_match_oracle(gpu, cfg, scale, triples):
    from oracle.ccsd_oracle import unpack_t2
    from oracle.triples_oracle import OracleTriples
    inp, oc = _pair(cfg)
    o, v = inp.nocc, inp.nvir
    t1, t2p = ci.random_amplitudes(o, v, 33, scale)
    ot = OracleTriples(oc, t1=t1, t2=unpack_t2(t2p, o, v))
    gc = gpu.CCSD(inp.h, inp.B, o, v)
    gc.set_amplitudes(t1, t2p)
    for (i, j, k) in triples:
        Wg, Zg, Yg = (x.cpu().numpy() for x in gc.triples_block(i, j, k))
        assert _rel(Wg, ot.W(i, j, k)[1]) <= REL_TOL, ("W", i, j, k)
        assert _rel(Zg, ot.Z(i, j, k)[1]) <= REL_TOL, ("Z", i, j, k)
        assert _rel(Yg, ot.Y(i, j, k)[1]) <= REL_TOL, ("Y", i, j, k)
    gc.close()


@pytest.mark.parametrize("cfg,scale", [("cfg0", 0.2), ("ragged", 0.05), ("ragged_even", 0.05)])
def test_triples_energies_match_oracle(gpu, cfg, scale):
    from oracle.ccsd_oracle import unpack_t2
    from oracle.triples_oracle import OracleTriples
    inp, oc = _pair(cfg)
    o, v = inp.nocc, inp.nvir
    gc = gpu.CCSD(inp.h, inp.B, o, v)
    # (a) seeded random amplitudes, (b) the CCSD iterate after three oracle iterations
    t1, t2p = ci.random_amplitudes(o, v, 34, scale)
    cases = [(t1, unpack_t2(t2p, o, v), t2p)]
    for _ in range(3):
        oc.iterate()
    from oracle.ccsd_oracle import pack_t2
    cases.append((oc.t1.copy(), oc.t2.copy(), pack_t2(oc.t2)))
    for a1, a2, a2p in cases:
        ref = OracleTriples(oc, t1=a1, t2=a2).energies(restricted=True)
        gc.set_amplitudes(a1, a2p)
        got = gc.triples()
        for key in ("+T", "(T)", "-T"):
            assert abs(got[key] - ref[key]) < E_TOL, (key, got[key], ref[key])
        assert abs(ref["+T"]) > 1e-9
    gc.close()


def test_triples_energies_cfg1_against_oracle_golden(gpu):
    """cfg1 (16/96): 560 occupied triples; the oracle needs minutes, so its energies at the seeded amplitudes
    CN(0, 0.01^2) (seed 35) are stored by tests/golden/make_oracle_triples.py (oracle/ only)."""
    path = os.path.join(GOLDEN, "oracle_triples_cfg1.txt")
    if not os.path.exists(path):
        pytest.skip(f"{path} not generated")
    ref = {}
    with open(path) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            key, re, im = line.split()
            ref[key] = complex(float(re), float(im))
    inp = ci.make_config("cfg1")
    o, v = inp.nocc, inp.nvir
    t1, t2p = ci.random_amplitudes(o, v, 35, 0.01)
    gc = gpu.CCSD(inp.h, inp.B, o, v)
    gc.set_amplitudes(t1, t2p)
    got = gc.triples()
    for key in ("+T", "(T)", "-T"):
        assert abs(got[key] - ref[key]) < E_TOL, (key, got[key], ref[key])
    gc.close()


def test_triples_edge_cases(gpu):
    """Degenerate sizes: fewer than three occupied spinors -> CCSD_EINVAL; exactly three occupied and three virtual
    spinors (ONE occupied triple, ONE virtual triple); level-shifted denominators; the call leaves the amplitudes and a
    following iteration untouched."""
    from paper_2103_08473_b200.binding import CCSDError
    from oracle.ccsd_oracle import OracleCCSD, pack_t2
    from oracle.triples_oracle import OracleTriples
    inp = ci.make_config("cfg0_2e")
    gc = gpu.CCSD(inp.h, inp.B, inp.nocc, inp.nvir)
    with pytest.raises(CCSDError):
        gc.triples()
    gc.close()
    inp = ci.make_inputs(3, 3, 5, seed=31, b_scale=0.2, f_offdiag=0.1)
    oc = OracleCCSD(inp.h, inp.B, 3, 3)
    gc = gpu.CCSD(inp.h, inp.B, 3, 3)
    oc.iterate(); gc.iterate()
    ref, got = OracleTriples(oc).energies(), gc.triples()
    for key in ("+T", "(T)", "-T"):
        assert abs(got[key] - ref[key]) < E_TOL and abs(ref[key]) > 1e-8, (key, got[key], ref[key])
    e_o, e_g = oc.iterate()[0], gc.iterate()[0]          # the triples call did not disturb the solver state
    assert abs(e_o - e_g) < E_TOL
    gc.close()
    inp = ci.make_inputs(5, 12, 20, seed=32)
    oc = OracleCCSD(inp.h, inp.B, 5, 12, level_shift=0.3)
    gc = gpu.CCSD(inp.h, inp.B, 5, 12, level_shift=0.3)
    for _ in range(2):
        oc.iterate(); gc.iterate()
    ref, got = OracleTriples(oc).energies(restricted=True), gc.triples()
    for key in ("+T", "(T)", "-T"):
        assert abs(got[key] - ref[key]) < E_TOL, (key, got[key], ref[key])
    gc.close()


def test_triples_do_not_depend_on_the_level_shift(gpu):
    """Converged with shift 0 and with shift 0.3 the amplitudes agree, so +T / (T) / -T must too: their denominators are the
    spinor energies Re f_pp, not the shifted ones of the Jacobi step (PAPER.md:1062 vs eqs 39/41).  Against the oracle too."""
    from oracle.ccsd_oracle import OracleCCSD
    from oracle.triples_oracle import OracleTriples
    o, v = 5, 11
    inp = ci.make_inputs(o, v, 18, seed=882, b_scale=0.1, f_offdiag=0.05)
    oc = OracleCCSD(inp.h, inp.B, o, v)
    assert oc.run(300, tol=1e-13)[-1][1] < 1e-12
    ref = OracleTriples(oc).energies(restricted=True)
    got = {}
    for shift in (0.0, 0.3):
        gc = gpu.CCSD(inp.h, inp.B, o, v, level_shift=shift)
        ok, nit, e, sn = gc.solve(1e-13, 600)
        assert ok, (shift, nit, sn)
        got[shift] = gc.triples()
        gc.close()
    for key in ("+T", "(T)", "-T"):
        assert abs(ref[key]) > 1e-7
        assert abs(got[0.0][key] - got[0.3][key]) < E_TOL, (key, got[0.0][key], got[0.3][key])
        assert abs(got[0.3][key] - ref[key]) < E_TOL, (key, got[0.3][key], ref[key])


@pytest.mark.parametrize("gemm_mode", [1, 2, 3])
def test_triples_and_cc2_under_every_gemm_mode(gpu, gemm_mode):
    """Triples (the K-segmented GEMM always runs on the DMMA kernel; without sum planes when they are switched off) and
    one CC2 iteration with the GEMM family forced."""
    from oracle.ccsd_oracle import OracleCCSD, pack_t2
    from oracle.cc2_oracle import OracleCC2
    from oracle.triples_oracle import OracleTriples
    inp = ci.make_inputs(5, 12, 20, seed=4720)
    o, v = inp.nocc, inp.nvir
    oc = OracleCCSD(inp.h, inp.B, o, v)
    for _ in range(3):
        oc.iterate()
    gc = gpu.CCSD(inp.h, inp.B, o, v, gemm_mode=gemm_mode)
    gc.set_amplitudes(oc.t1, pack_t2(oc.t2))
    ref, got = OracleTriples(oc).energies(restricted=True), gc.triples()
    for key in ("+T", "(T)", "-T"):
        assert abs(got[key] - ref[key]) < E_TOL, (key, got[key], ref[key])
    gc.close()
    o2 = OracleCC2(inp.h, inp.B, o, v)
    g2 = gpu.CCSD(inp.h, inp.B, o, v, gemm_mode=gemm_mode, cc2=True)
    for _ in range(3):
        eo, eg = o2.iterate()[0], g2.iterate()[0]
        assert abs(eo - eg) < E_TOL
    g2.close()


def test_triples_ranges_match_oracle_partial_sums(gpu):
    """ccsd_triples_range (the unit of the multi-GPU split): partial sums over ranges of the lexicographic list of i<j<k
    against the oracle's partial sums over the same triples; the pieces of every partition add up to ccsd_triples."""
    import itertools
    from paper_2103_08473_b200.binding import CCSDError
    from paper_2103_08473_b200.sharding import shard_range
    from oracle.ccsd_oracle import OracleCCSD
    from oracle.triples_oracle import OracleTriples
    o, v = 6, 9
    inp = ci.make_inputs(o, v, 14, seed=61, b_scale=0.15, f_offdiag=0.05)
    oc = OracleCCSD(inp.h, inp.B, o, v)
    gc = gpu.CCSD(inp.h, inp.B, o, v)
    for _ in range(2):
        oc.iterate(); gc.iterate()
    ot = OracleTriples(oc)
    triples = list(itertools.combinations(range(o), 3))
    assert gc.triples_count() == len(triples) == 20
    full = gc.triples()
    for world in (1, 2, 3, 7):
        tot = {"+T": 0.0, "(T)": 0.0, "-T": 0.0}
        for rank in range(world):
            first, count = shard_range(len(triples), rank, world)
            got = gc.triples_range(first, count)
            ref = ot.energies_of(triples[first:first + count])
            for key in tot:
                assert abs(got[key] - ref[key]) < E_TOL, (world, rank, key, got[key], ref[key])
                tot[key] += got[key]
        for key in tot:
            assert abs(tot[key] - full[key]) < 1e-13, (world, key)
    empty = gc.triples_range(20, 0)
    assert all(empty[key] == 0 for key in empty)
    assert gc.triples_sharded() == full                  # no process group: the whole list on this GPU
    for first, count in ((-1, 2), (0, 21), (20, 1), (3, -1)):
        with pytest.raises(CCSDError):
            gc.triples_range(first, count)
    gc.close()
