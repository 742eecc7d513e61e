"""GPU parity of the Strassen level (csrc/strassen.cuh; ccsd_options.strassen, ccsd_zgemm_nt_strassen): the seven-product form
must equal the plain definition C = alpha A B^T (+ C) within the 1e-12 relative (max-abs) bound of BASELINE.json's north_star.

* ccsd_zgemm_nt_strassen against numpy's complex128 matmul on the host, element by element: odd and even extents (the odd
  halves are zero-padded inside the operand stacks), both output orders, complex alpha, accumulation, extents of 1;
* a context with strassen = 1 against the same context with strassen = 0 at a size where the level is used (cfg1: ov = 1536):
  every intermediate, every term of eq 32, S1, S2 and the lock-step energies;
* the lock-step / converged-energy tests of test_gpu_parity.py and test_gpu_fullsize.py run with the default (strassen = 1) at
  cfg1, cfg2, cfg3 against the oracle; sizes below ov = 1024 (cfg0 and the ragged shapes) keep exercising the plain products.
"""
import numpy as np
import pytest

import ccsd_inputs as ci

pytestmark = pytest.mark.gpu

REL_TOL = 1e-12


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2103_08473_b200 as lib
    lib.load_library()
    return lib


def _rand(shape, seed, scale=1.0):
    rng = np.random.default_rng(seed)
    return scale * (rng.standard_normal(shape) + 1j * rng.standard_normal(shape))


def _rel(a, b):
    scale = np.abs(b).max()
    return np.abs(np.asarray(a) - np.asarray(b)).max() / (scale if scale > 0 else 1.0)


@pytest.mark.parametrize("M,N,K", [(1031, 97, 1033), (1024, 96, 1024), (257, 129, 515), (130, 50, 70), (5, 3, 7), (2, 2, 2),
                                   (1, 1, 1), (1, 9, 4), (300, 1, 33), (64, 64, 1), (7, 6, 5), (3, 3, 3), (515, 262, 1031)])
@pytest.mark.parametrize("transposed_out", [False, True])
@pytest.mark.parametrize("levels", [1, 2])
def test_strassen_gemm_equals_the_definition(gpu, M, N, K, transposed_out, levels):
    import torch
    A, B = _rand((M, K), 10 * M + K), _rand((N, K), 10 * N + K + 1)
    want = A @ B.T
    got = gpu.zgemm_nt_strassen(A, B, transposed_out=transposed_out, levels=levels).cpu().numpy()
    got = got.T if transposed_out else got
    assert _rel(got, want) < REL_TOL, _rel(got, want)
    # complex alpha, accumulation into a non-zero C (the products' scratch still holds the previous call's values)
    alpha = 0.7 - 1.3j
    C0 = _rand((N, M) if transposed_out else (M, N), 77)
    C = torch.from_numpy(C0.copy()).cuda()
    gpu.zgemm_nt_strassen(A, B, C=C, alpha=alpha, accumulate=True, transposed_out=transposed_out, levels=levels)
    got = C.cpu().numpy()
    ref = (C0.T if transposed_out else C0) + alpha * want
    assert _rel(got.T if transposed_out else got, ref) < REL_TOL


@pytest.mark.parametrize("M,N,K,transposed_out", [(3840, 3840, 3840, False), (12720, 276, 12720, True)])
def test_strassen_error_against_extended_precision_sums(gpu, M, N, K, transposed_out):
    """The error claim of DESIGN.md "Strassen levels" at sizes where the levels are used (cfg2's (ov)^3 and ladder shapes): sampled
    elements against 80-bit sums formed on the host.  Plain 3M product and one / two levels all stay below 5e-14 of the largest
    element of C -- a factor 20 inside the 1e-12 parity bound -- and the levels lose at most a factor 4 on the plain product."""
    import torch
    g = torch.Generator(device="cuda"); g.manual_seed(M + N)
    A = torch.view_as_complex(torch.randn(M, K, 2, dtype=torch.float64, device="cuda", generator=g))
    B = torch.view_as_complex(torch.randn(N, K, 2, dtype=torch.float64, device="cuda", generator=g))
    rng = np.random.default_rng(3)
    ms, ns = rng.integers(0, M, 96), rng.integers(0, N, 96)
    Ah, Bh = A[torch.from_numpy(ms).cuda()].cpu().numpy(), B[torch.from_numpy(ns).cuda()].cpu().numpy()
    ar, ai, br, bi = [x.astype(np.longdouble) for x in (Ah.real, Ah.imag, Bh.real, Bh.imag)]
    ex_re, ex_im = (ar * br - ai * bi).sum(1), (ar * bi + ai * br).sum(1)

    def err(C):
        Cf = C.t() if transposed_out else C
        x = Cf[torch.from_numpy(ms).cuda(), torch.from_numpy(ns).cuda()].cpu().numpy()
        scale = float(C.abs().max())
        return float(max(np.abs(x.real - ex_re).max(), np.abs(x.imag - ex_im).max())) / scale

    e0 = err(gpu.zgemm_nt(A, B, transposed_out=transposed_out))
    e1 = err(gpu.zgemm_nt_strassen(A, B, transposed_out=transposed_out, levels=1))
    e2 = err(gpu.zgemm_nt_strassen(A, B, transposed_out=transposed_out, levels=2))
    assert e0 < 5e-14 and e1 < 5e-14 and e2 < 5e-14, (e0, e1, e2)
    assert e1 < 4 * e0 + 1e-15 and e2 < 4 * e0 + 1e-15, (e0, e1, e2)


def test_strassen_gemm_equals_the_plain_dmma_gemm_at_a_ladder_like_shape(gpu):
    """(a<b) x (i<j) x (c<d) with an odd N, output transposed as the pp-ladder writes it; sampled rows against numpy."""
    import torch
    M, N, K = 4560, 121, 4560
    g = torch.Generator(device="cuda"); g.manual_seed(5)
    A = torch.view_as_complex(torch.randn(M, K, 2, dtype=torch.float64, device="cuda", generator=g))
    B = torch.view_as_complex(torch.randn(N, K, 2, dtype=torch.float64, device="cuda", generator=g))
    plain = gpu.zgemm_nt(A, B, transposed_out=True)
    scale = float(plain.abs().max())
    rows = [0, 1, 1139, 1140, 1141, 2279, 2280, 2281, 3419, 3420, 3421, 4559]      # both sides of every split
    want = (A[rows].cpu().numpy() @ B.cpu().numpy().T).T                           # [n][rows]
    for levels in (1, 2):
        fast = gpu.zgemm_nt_strassen(A, B, transposed_out=True, levels=levels)
        assert float((plain - fast).abs().max()) / scale < 1e-13
        assert np.abs(fast[:, rows].cpu().numpy() - want).max() / scale < REL_TOL


@pytest.mark.parametrize("mode", [1, 2, 3])
def test_context_with_strassen_equals_context_without(gpu, mode):
    """cfg1 (16/96/336): ov = 1536, vv = 4560 -- the scheme is used for the two (ov)^3 products and the pp-ladder.  mode 1: the
    default choice of levels (one, at this size), 2: one level, 3: two levels forced on all four products (the packed <ab||cd> is
    then kept as the ladder's operand stack only)."""
    o, v, naux = 16, 96, 336
    inp = ci.make_inputs(o, v, naux, 2021030801)
    fast = gpu.CCSD(inp.h, inp.B, o, v, strassen=mode)
    plain = gpu.CCSD(inp.h, inp.B, o, v, strassen=0)
    assert fast.workspace_bytes > plain.workspace_bytes      # the operand stacks of the constants
    assert fast.strassen_steps().get("ring_gemm") == (2 if mode == 3 else 1) and plain.strassen_steps() == {}
    # same (MP2) amplitudes in both: every product on its own scale; the sums S1, S2 cancel against the driver term, so they
    # get the north_star bound relative to the largest term
    fast.residual(); plain.residual()
    term_scale = 0.0
    for name in ["tau", "Hvovo", "C", "A", "S2_pp_ladder", "S2_ring", "S2_hh_ladder", "S2_c_t1", "S2_driver"]:
        a, b = fast.get_tensor(name).cpu().numpy(), plain.get_tensor(name).cpu().numpy()
        assert _rel(a, b) < 1e-13, (name, _rel(a, b))
        if name.startswith("S2_"):
            term_scale = max(term_scale, np.abs(b).max())
    for name in ["S1", "S2"]:
        a, b = fast.get_tensor(name).cpu().numpy(), plain.get_tensor(name).cpu().numpy()
        assert np.abs(a - b).max() < REL_TOL * max(term_scale, np.abs(b).max()), name
    a, b = fast.get_tensor("vvvv").cpu().numpy(), plain.get_tensor("vvvv").cpu().numpy()
    assert _rel(a, b) < 4e-16                  # stored tensor / rebuilt from the ladder's operand stack: one rounding at most
    for it in range(4):
        ef, nf = fast.iterate()
        ep, npl = plain.iterate()
        assert abs(ef - ep) < 1e-12 * max(1.0, abs(ep)), (it, ef, ep)
        assert abs(nf - npl) < 1e-10 * max(npl, 1e-6)
    fast.close(); plain.close()
