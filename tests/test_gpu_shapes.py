"""GPU parity at occupied-heavy shapes: more occupied spinors than one 48-column GEMM tile, and more occupied than virtual
spinors (the scratch of the Lambda path is then sized by o^4, not by o v^3).  CCSD lock-step, the triples energies, the
Lambda right-hand sides / density at seeded random multipliers and the standalone intermediates, each against its oracle
at identical amplitudes.  Tolerances as everywhere: 1e-12 relative max-abs per tensor, 1e-10 Eh on energies."""
import numpy as np
import pytest

import ccsd_inputs as ci

pytestmark = pytest.mark.gpu


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
    return np.abs(np.asarray(a).ravel() - np.asarray(b).ravel()).max() / (scale if scale > 0 else 1.0)


@pytest.mark.parametrize("o,v,L,b_scale", [(52, 7, 12, 0.1), (50, 20, 30, 0.03)])
def test_occupied_heavy_shapes(gpu, o, v, L, b_scale):
    from oracle.ccsd_oracle import OracleCCSD, pack_t2, unpack_t2
    from oracle.lambda_oracle import OracleLambda
    from oracle.triples_oracle import OracleTriples
    inp = ci.make_inputs(o, v, L, seed=100 + o + v, b_scale=b_scale, f_offdiag=0.05)
    oc = OracleCCSD(inp.h, inp.B, o, v)
    gc = gpu.CCSD(inp.h, inp.B, o, v)
    for _ in range(3):
        (eo, so), (eg, sg) = oc.iterate(), gc.iterate()
        assert abs(eo - eg) < 1e-10 and abs(so - sg) < 1e-11 * max(1.0, so)
    # triples at the oracle's amplitudes
    gc.set_amplitudes(oc.t1, pack_t2(oc.t2))
    ref, got = OracleTriples(oc).energies(restricted=True), gc.triples()
    for key in ref:
        assert abs(ref[key] - got[key]) < 1e-10 * max(1.0, abs(ref[key])), (key, ref[key], got[key])
    assert abs(ref["+T"]) > 1e-6
    # Lambda right-hand sides and density at seeded random multipliers
    ol = OracleLambda(oc)
    gc.lambda_init()
    l1, l2p = ci.random_amplitudes(o, v, 44, 0.2)
    gc.set_lambda(l1, l2p)
    R1, R2 = ol.residual(l1, unpack_t2(l2p, o, v))
    r1, r2p = gc.lambda_residual()
    assert _rel(r1.cpu().numpy(), R1) < 1e-12 and _rel(r2p.cpu().numpy(), pack_t2(R2)) < 1e-12
    assert _rel(gc.density().cpu().numpy(), ol.density(l1, unpack_t2(l2p, o, v))) < 1e-12
    gc.close()
    # the standalone intermediates (their scratch is sized the same way)
    oc.build_intermediates()
    io, jo = np.triu_indices(o, 1)
    av, bv = np.triu_indices(v, 1)
    can = {"oooo": oc.oooo[io[:, None], jo[:, None], io[None, :], jo[None, :]], "ooov": oc.ooov[io, jo],
           "oovv": oc.oovv[io[:, None], jo[:, None], av[None, :], bv[None, :]], "t1": oc.t1, "t2": pack_t2(oc.t2)}
    can = {k: np.ascontiguousarray(x) for k, x in can.items()}
    A = gpu.contract("w_oooo", o, v, [can[k] for k in ("oooo", "ooov", "oovv", "t1", "t2")]).cpu().numpy()
    assert _rel(A, oc.A[io[:, None], jo[:, None], io[None, :], jo[None, :]]) < 1e-12


def test_dmma_pipeline_is_race_free_by_determinism_under_stress(gpu):
    """compute-sanitizer (racecheck / synccheck) is closed on the GPU pool, so the hand-rolled TMA + full/empty mbarrier ring
    with its rotating issuer (gemm_dmma.cuh) is checked the other way round: a race in the ring (a stage overwritten before
    every warp released it, a fragment read before its copy landed) shows up as a run-to-run difference.  Every launch
    family -- 4M, 3M, 3M with sum planes, wide 4-d maps (K % 4 == 0) and 3-d maps (ragged K), split-K (no workspace ->
    none here; the in-context launches cover it), batched, accumulate -- is repeated 25 times while a second stream keeps
    the SMs and the memory system busy: all results must be BIT-identical, and equal to the simple FMA kernel to 1e-12."""
    import torch
    rng = np.random.default_rng(7)

    def cmat(m, k):
        return torch.from_numpy((rng.standard_normal((m, k)) + 1j * rng.standard_normal((m, k))) * 0.1).cuda()

    side = torch.cuda.Stream()
    noise_a = torch.randn(4096, 4096, device="cuda", dtype=torch.float64)
    shapes = [(300, 70, 16 * 37), (257, 48, 16 * 21 + 7), (128, 100, 64), (513, 34, 224), (640, 96, 1000)]
    for (M, N, K) in shapes:
        A, B = cmat(M, K), cmat(N, K)
        ref = gpu.zgemm_nt(A, B, mode=1)
        planes = (gpu.sum_plane(A), gpu.sum_plane(B)) if K % 2 == 0 else None
        for mode, pl in ((2, None), (3, None), (3, planes), (0, planes)):
            if mode == 0 and pl is None:
                continue
            first = None
            for rep in range(25):
                with torch.cuda.stream(side):
                    torch.matmul(noise_a, noise_a)                        # concurrent load on the other stream
                C = gpu.zgemm_nt(A, B, mode=mode, planes=pl, transposed_out=bool(rep & 1))
                C = C.t() if rep & 1 else C
                if first is None:
                    first = C.clone()
                    assert _rel(first.cpu().numpy(), ref.cpu().numpy()) < 1e-12, (M, N, K, mode)
                else:
                    assert torch.equal(C, first), (M, N, K, mode, rep)
            # accumulate path (prefetched read-modify-write epilogue)
            acc0 = cmat(M, N)
            outs = []
            for rep in range(10):
                Cacc = acc0.clone()
                gpu.zgemm_nt(A, B, C=Cacc, accumulate=True, mode=mode, planes=pl)
                outs.append(Cacc)
            assert all(torch.equal(outs[0], x) for x in outs[1:]), (M, N, K, mode)
            assert _rel((outs[0] - acc0).cpu().numpy(), ref.cpu().numpy()) < 1e-12
    side.synchronize()
    # the K-segmented loader of the triples and the whole iteration (split-K, batched launches, graph replay): repeated runs
    inp = ci.make_inputs(7, 26, 40, seed=91, b_scale=0.06)
    runs = []
    for rep in range(4):
        gc = gpu.CCSD(inp.h, inp.B, inp.nocc, inp.nvir)
        hist = [gc.iterate() for _ in range(6)]
        with torch.cuda.stream(side):
            torch.matmul(noise_a, noise_a)
        trip = gc.triples()
        W = gc.triples_block(1, 3, 5)[0].clone()
        runs.append((hist, trip, W))
        gc.close()
    for hist, trip, W in runs[1:]:
        assert hist == runs[0][0] and trip == runs[0][1] and torch.equal(W, runs[0][2])
