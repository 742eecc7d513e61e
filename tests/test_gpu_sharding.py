"""Slab sharding of the CCSD iteration (ccsd_options.shard_rank / shard_world) checked on ONE GPU: the P
contexts "rank r of P" are created one after the other on the same device and amplitudes.  Their slabs of every term of
eq 32 tile the single-GPU term (disjoint supports for the ladder term, equal there to rounding), the slabs of S2 add up to the
single-GPU S2 and to the oracle's, and residual -> sum over ranks -> ccsd_update reproduces ccsd_iterate step by step.
The all-reduce itself (torch.distributed) is covered by the world-2 gloo test on CPU (tests/test_sharding_cpu.py).
Unmeasured on more than one GPU: this pool has one."""
import numpy as np
import pytest

import ccsd_inputs as ci

pytestmark = pytest.mark.gpu

REL_TOL = 1e-12
E_TOL = 1e-10


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2103_08473_b200 as lib
    lib.load_library()
    return lib


def _rel(a, b):
    scale = float(np.abs(b).max())
    return float(np.abs(a - b).max()) / (scale if scale > 0 else 1.0)


@pytest.mark.parametrize("o,v,naux,direct,strassen", [(6, 21, 30, False, 1), (9, 40, 50, False, 1), (5, 17, 24, True, 1),
                                                      (6, 21, 30, False, 3), (9, 40, 50, False, 3), (5, 17, 24, True, 3)])
def test_slabs_tile_the_single_gpu_residual_and_match_the_oracle(gpu, o, v, naux, direct, strassen):
    """strassen = 3: two Strassen levels forced on every rank's slab products (left operands = the rank's row slabs, odd and empty
    slabs included), the rank's rows of <ab||cd> kept as their operand stack only."""
    import torch
    from oracle.ccsd_oracle import OracleCCSD, pack_t2, unpack_t2
    inp = ci.make_inputs(o, v, naux, seed=5200 + o + v, b_scale=0.08, f_offdiag=0.05)
    t1, t2p = ci.random_amplitudes(o, v, 53, 0.05)
    oc = OracleCCSD(inp.h, inp.B, o, v)
    oc.set_amplitudes(t1, unpack_t2(t2p, o, v))
    S1o, S2o = oc.residual()
    S2o = pack_t2(S2o)
    one = gpu.CCSD(inp.h, inp.B, o, v, direct_ladder=direct, strassen=strassen)
    one.set_amplitudes(t1, t2p)
    one.residual()
    full = {name: one.get_tensor(name).clone() for name in ("S2", "S1", "S2_pp_ladder", "S2_ring", "S2_hh_ladder", "S2_goo",
                                                             "S2_vdag_t1", "S2_gvv", "S2_c_t1", "S2_driver", "Hvovo", "C")}
    one.close()
    assert _rel(full["S2"].cpu().numpy().reshape(S2o.shape), S2o) <= REL_TOL
    for world in (1, 2, 3, 7):
        acc = {k: torch.zeros_like(x) for k, x in full.items() if k.startswith("S2")}
        support = torch.zeros_like(full["S2_pp_ladder"], dtype=torch.int32)
        for rank in range(world):
            gc = gpu.CCSD(inp.h, inp.B, o, v, shard=(rank, world), direct_ladder=direct, strassen=strassen)
            if strassen == 3 and (info_rows := gc.shard_info()) and info_rows["a_hi"] > info_rows["a_lo"]:
                assert gc.strassen_steps().get("ring_gemm") == 2
            info = gc.shard_info()
            assert (info["rank"], info["world"]) == (rank, world)
            assert gc.workspace_bytes <= one.workspace_bytes
            gc.set_amplitudes(t1, t2p)
            gc.residual()
            assert _rel(gc.get_tensor("S1").cpu().numpy(), full["S1"].cpu().numpy()) <= 1e-14      # replicated
            assert torch.equal(gc.s2_view().reshape(-1), gc.get_tensor("S2"))                      # the view IS the buffer
            for name in acc:
                part = gc.get_tensor(name)
                acc[name] += part
                if name == "S2_pp_ladder":      # disjoint (a<b) column slabs, equal to the single-GPU term there (the split-K
                    nz = part != 0              # depth, hence the summation order, depends on the number of row tiles)
                    support += nz.to(torch.int32)
                    assert float((part[nz] - full[name][nz]).abs().max()) <= 1e-13 * float(full[name].abs().max())
                    cols = nz.view(gc.oo, gc.vv).any(dim=0).nonzero().flatten()
                    if len(cols):
                        assert info["w_lo"] <= int(cols.min()) and int(cols.max()) < info["w_hi"]
            # rows of H^{ak}_{ci} and of C outside the slab are never touched by a sharded residual; inside they are exact
            H = gc.get_tensor("Hvovo").view(v, o, v, o)[info["a_lo"]:info["a_hi"]]
            Hf = full["Hvovo"].view(v, o, v, o)[info["a_lo"]:info["a_hi"]]
            assert float((H - Hf).abs().max()) <= 1e-13 * float(full["Hvovo"].abs().max())
            Cg = gc.get_tensor("C").view(o, v, -1)[:, info["a_lo"]:info["a_hi"]]
            Cf = full["C"].view(o, v, -1)[:, info["a_lo"]:info["a_hi"]]
            assert float((Cg - Cf).abs().max()) <= 1e-13 * float(full["C"].abs().max())
            if world > 1:
                from paper_2103_08473_b200.binding import CCSDError
                with pytest.raises(CCSDError):
                    gc.solve(1e-9, 3)                       # ccsd_iterate / ccsd_solve need the caller's all-reduce
            gc.close()
        assert int(support.max()) <= 1
        for name, x in acc.items():
            assert _rel(x.cpu().numpy(), full[name].cpu().numpy()) <= 1e-13, (world, name)
        assert _rel(acc["S2"].cpu().numpy().reshape(S2o.shape), S2o) <= REL_TOL, world


@pytest.mark.parametrize("strassen", [1, 3])
def test_sharded_iteration_protocol_reproduces_ccsd_iterate(gpu, strassen):
    """residual on every rank -> sum of the S2 slabs written back into every rank's buffer (what the all-reduce does) ->
    ccsd_update on every rank: lock step with the single-GPU ccsd_iterate and with the oracle, DIIS included; every rank ends
    each iteration with identical amplitudes."""
    import torch
    from oracle.ccsd_oracle import OracleCCSD
    o, v, world = 6, 22, 3
    inp = ci.make_inputs(o, v, 36, seed=5300, b_scale=0.1, f_offdiag=0.05)
    oc = OracleCCSD(inp.h, inp.B, o, v)
    one = gpu.CCSD(inp.h, inp.B, o, v, strassen=strassen)
    ranks = [gpu.CCSD(inp.h, inp.B, o, v, shard=(r, world), strassen=strassen) for r in range(world)]
    for it in range(9):
        eo, so = oc.iterate()
        e1, s1 = one.iterate()
        for g in ranks:
            g.residual()
        total = sum(g.s2_view().clone() for g in ranks)
        outs = []
        for g in ranks:
            g.s2_view().copy_(total)
            outs.append(g.update())
        assert all(x == outs[0] for x in outs), (it, outs)
        assert abs(outs[0][0] - e1) < 1e-12 and abs(outs[0][0] - eo) < E_TOL, (it, outs[0], e1, eo)
        assert abs(outs[0][1] - so) < 1e-9 * max(1.0, so)
        amps = [g.get_amplitudes() for g in ranks]
        assert all(torch.equal(a[0], amps[0][0]) and torch.equal(a[1], amps[0][1]) for a in amps)
    for g in ranks + [one]:
        g.close()


def test_sharded_context_without_a_process_group_iterates_alone(gpu):
    """CCSD.iterate in a sharded context = residual + all-reduce + update; without an initialised process group the
    all-reduce is a no-op, so world = 1 through that path equals the plain iteration."""
    inp = ci.make_config("cfg0")
    a = gpu.CCSD(inp.h, inp.B, inp.nocc, inp.nvir)
    b = gpu.CCSD(inp.h, inp.B, inp.nocc, inp.nvir, shard=(0, 1))
    from paper_2103_08473_b200.sharding import iterate_sharded
    for _ in range(4):
        assert a.iterate() == iterate_sharded(b)
    a.close(); b.close()
