"""ccsd_energy_static (include/ccsd.h): the correlation energy of eq 9 (tau of eq 23) through the entry point
that takes no workspace -- its scratch (pair tables, per-block partial sums) is a fixed device array inside the library --
against the existing workspace path ccsd_contract(CCSD_TERM_ENERGY) on the same inputs, on calls in a row that share that
array, and against the definition written out with numpy.  Collected last on purpose (the name): the suite runs with
pytest -x.  Needs no state from other tests: passes alone in a fresh process and after the rest of the suite.
"""
import ctypes

import numpy as np
import pytest

import ccsd_inputs as ci

TOL = 1e-12          # the tolerance tests/test_gpu_terms.py uses for the energy term


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2103_08473_b200 as lib
    lib.load_library()
    return lib


def _inputs(o, v, seed):
    """Seeded synthetic operands of eq 9 in the boundary layouts: f [n][n], <kl||cd> [(k<l)][(c<d)], t1 [i][a], t2 packed."""
    rng = np.random.default_rng(seed)
    n, oo, vv = o + v, o * (o - 1) // 2, v * (v - 1) // 2
    f = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    oovv = 0.1 * (rng.standard_normal((oo, vv)) + 1j * rng.standard_normal((oo, vv)))
    t1, t2p = ci.random_amplitudes(o, v, seed + 1, 0.3)
    return [np.ascontiguousarray(x, dtype=np.complex128) for x in (f, oovv, t1, t2p)]


def _definition(o, v, f, oovv, t1, t2p):
    """E = sum_ia f_ia t^a_i + sum_{i<j,a<b} <ij||ab> (t2 + t1 t1 - t1 t1)^{ab}_{ij}, eq 9 with tau of eq 23."""
    i, j = np.triu_indices(o, 1)
    a, b = np.triu_indices(v, 1)
    tau = t2p + t1[i][:, a] * t1[j][:, b] - t1[j][:, a] * t1[i][:, b]
    return (f[:o, o:] * t1).sum() + (oovv * tau).sum()


@pytest.mark.gpu
def test_energy_static_equals_the_workspace_path_on_calls_in_a_row(gpu):
    import torch
    # (o, v, seed): several 1024-column tiles with a ragged tail; the same shape again with other amplitudes; a small shape
    # AFTER a large one (the shared tables and partials still hold the large call's contents); more tiles than blocks
    cases = [(7, 60, 11), (7, 60, 12), (4, 6, 13), (2, 2, 14), (12, 150, 15), (5, 9, 16)]
    dev = [[torch.from_numpy(x).cuda() for x in _inputs(o, v, seed)] for (o, v, seed) in cases]
    outs = [torch.full((1,), 7.0 + 7.0j, dtype=torch.complex128, device="cuda") for _ in cases]   # must be OVERWRITTEN
    want = [gpu.contract("energy", o, v, d).cpu().numpy()[0] for (o, v, _), d in zip(cases, dev)]  # the existing path
    torch.cuda.synchronize()

    gpu.energy_static(cases[0][0], cases[0][1], *dev[0], outs[0])      # first call on this device resolves the address
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    for (o, v, _), d, out in zip(cases[1:], dev[1:], outs[1:]):        # back to back on one stream, no sync between them
        gpu.energy_static(o, v, *d, out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before                 # nothing was allocated on the device

    for (o, v, seed), d, out, w in zip(cases, dev, outs, want):
        got = out.cpu().numpy()[0]
        ref = _definition(o, v, *[x.cpu().numpy() for x in d])
        assert abs(w - ref) < TOL * max(1.0, abs(ref)), (o, v, w, ref)
        assert abs(got - w) < TOL * max(1.0, abs(w)), (o, v, got, w)
        assert got == w, (o, v, got, w)                                # same kernels, same summation order: same bits

    # the whole sequence once more: results must not depend on what the previous calls left in the scratch
    for (o, v, _), d, out, w in zip(cases, dev, outs, want):
        out.fill_(-3.0)
        gpu.energy_static(o, v, *d, out)
        assert out.cpu().numpy()[0] == w


@pytest.mark.gpu
def test_energy_static_equals_the_oracle_energy(gpu):
    import torch
    from oracle.ccsd_oracle import OracleCCSD, pack_t2, unpack_t2
    o, v = 5, 11
    inp = ci.make_inputs(o, v, 17, 62, b_scale=0.1, f_offdiag=0.05)
    oc = OracleCCSD(inp.h, inp.B, o, v)
    t1, t2p = ci.random_amplitudes(o, v, 63, scale=0.05)
    oc.set_amplitudes(t1, unpack_t2(t2p, o, v))
    io, jo = np.triu_indices(o, 1)
    av, bv = np.triu_indices(v, 1)
    ins = [oc.f, oc.oovv[io[:, None], jo[:, None], av[None, :], bv[None, :]], oc.t1, pack_t2(oc.t2)]
    dev = [torch.from_numpy(np.ascontiguousarray(x, dtype=np.complex128)).cuda() for x in ins]
    out = torch.zeros(1, dtype=torch.complex128, device="cuda")
    for _ in range(2):
        e = gpu.energy_static(o, v, *dev, out).cpu().numpy()[0]
        want = oc.energy()
        assert abs(e - want) < TOL * max(1.0, abs(want)), (e, want)


@pytest.mark.gpu
def test_energy_static_rejects_sizes_beyond_its_scratch(gpu):
    import torch
    from paper_2103_08473_b200 import binding
    for o, v in ((binding.ENERGY_STATIC_MAX_NOCC + 1, 4), (2, binding.ENERGY_STATIC_MAX_NVIR + 1)):
        oo, vv = o * (o - 1) // 2, v * (v - 1) // 2
        z = lambda *s: torch.zeros(s, dtype=torch.complex128, device="cuda")
        out = torch.full((1,), 5.0 + 0j, dtype=torch.complex128, device="cuda")
        with pytest.raises(gpu.CCSDError) as err:
            gpu.energy_static(o, v, z(o + v, o + v), z(oo, vv), z(o, v), z(oo, vv), out)
        assert err.value.status == 1 and "beyond the static scratch" in str(err.value)      # CCSD_EINVAL, with the reason
        torch.cuda.synchronize()
        assert out.cpu().numpy()[0] == 5.0                                                  # nothing was enqueued
    # the limits themselves are accepted
    o, v = 3, binding.ENERGY_STATIC_MAX_NVIR
    ins = [torch.from_numpy(x).cuda() for x in _inputs(o, v, 21)]
    out = torch.zeros(1, dtype=torch.complex128, device="cuda")
    got = gpu.energy_static(o, v, *ins, out).cpu().numpy()[0]
    assert got == gpu.contract("energy", o, v, ins).cpu().numpy()[0]


def test_energy_static_limits_are_checked_before_any_cuda_call():
    """No GPU needed: the size and pointer checks come first, so they can be exercised on a CPU box."""
    from paper_2103_08473_b200 import binding
    lib = binding.load_library()
    buf = ctypes.create_string_buffer(64)      # never dereferenced: the call must return before touching it
    p = ctypes.addressof(buf)
    assert lib.ccsd_energy_static(binding.ENERGY_STATIC_MAX_NOCC + 1, 8, p, p, p, p, p, None) == 1
    assert b"beyond the static scratch" in lib.ccsd_last_cuda_error()
    assert lib.ccsd_energy_static(8, binding.ENERGY_STATIC_MAX_NVIR + 1, p, p, p, p, p, None) == 1
    assert lib.ccsd_energy_static(1, 8, p, p, p, p, p, None) == 1          # nocc, nvir >= 2 as for CCSD_TERM_ENERGY
    assert lib.ccsd_energy_static(8, 8, None, p, p, p, p, None) == 1       # null operand
    assert lib.ccsd_energy_static(8, 8, p, p, p, p, None, None) == 1       # null output
    # the documented size of the scratch: partials (2 per block of 592) + one 8-byte pair per (i<j) and per (a<b) at the limits
    mo, mv = binding.ENERGY_STATIC_MAX_NOCC, binding.ENERGY_STATIC_MAX_NVIR
    assert binding.ENERGY_STATIC_SCRATCH_BYTES == 8 * (2 * 592 + mo * (mo - 1) // 2 + mv * (mv - 1) // 2)
