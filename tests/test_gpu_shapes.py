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
