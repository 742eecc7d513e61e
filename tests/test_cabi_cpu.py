"""CPU-only checks of the boundary: the C-ABI library loads, exports every symbol include/ccsd.h declares, its host
logic (sizes, defaults, error codes) behaves, and nothing computes without a GPU (no CPU fallback)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2103_08473_b200 import build
    build.build()                       # nvcc cross-compiles for sm_100a without a GPU
    import paper_2103_08473_b200 as pkg
    return pkg.load_library()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "ccsd.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ccsd_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    names = declared_symbols()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), n
    from paper_2103_08473_b200.binding import EXPORTS
    assert sorted(EXPORTS) == names


def test_defaults_and_strerror(lib):
    from paper_2103_08473_b200.binding import Options
    o = Options()
    lib.ccsd_default_options(ctypes.byref(o))
    assert (o.ndiis, o.level_shift, o.gemm_mode, o.ccd, o.cc2, o.direct_ladder, o.graph) == (6, 0.0, 0, 0, 0, 0, 1)
    assert (o.shard_rank, o.shard_world, o.strassen) == (0, 1, 1)
    assert lib.ccsd_strerror(0) == b"ok"
    assert b"CUDA" in lib.ccsd_strerror(3)
    assert lib.ccsd_step_name(6) == b"pp_ladder" and lib.ccsd_step_name(99) == b""


def test_workspace_bytes_scales_and_validates(lib):
    n = ctypes.c_size_t(0)
    assert lib.ccsd_workspace_bytes(4, 16, 60, None, ctypes.byref(n)) == 0
    small = n.value
    assert lib.ccsd_workspace_bytes(34, 224, 774, None, ctypes.byref(n)) == 0
    big = n.value
    vv = 224 * 223 // 2
    assert big > 3 * vv * vv * 16 and big < 115 * 2 ** 30   # holds the two-level Strassen stack of <ab||cd> (3.06 x the tensor with planes); fits a 180 GB part with the Lambda workspace beside it
    from paper_2103_08473_b200.binding import _options
    plain = _options(strassen=False)
    assert lib.ccsd_workspace_bytes(34, 224, 774, ctypes.byref(plain), ctypes.byref(n)) == 0
    assert vv * vv * 16 < n.value < 80 * 2 ** 30 and n.value < big   # the operand stacks of the constants are what strassen costs
    assert small < big
    assert lib.ccsd_workspace_bytes(1, 16, 60, None, ctypes.byref(n)) == 1      # CCSD_EINVAL
    assert lib.ccsd_workspace_bytes(4, 16, 0, None, ctypes.byref(n)) == 1
    assert lib.ccsd_workspace_bytes(4, 16, 60, None, None) == 1
    assert lib.ccsd_contract_workspace_bytes(0, 4, 16, ctypes.byref(n)) == 0
    assert lib.ccsd_contract_workspace_bytes(7, 4, 16, ctypes.byref(n)) == 0      # F_OO
    assert lib.ccsd_contract_workspace_bytes(11, 4, 16, ctypes.byref(n)) == 0     # S1_RESIDUAL
    big_term = n.value
    assert lib.ccsd_contract_workspace_bytes(13, 4, 16, ctypes.byref(n)) == 0     # ENERGY: pair tables, tau, eps only
    assert 120 * 6 * 16 <= n.value < big_term
    assert lib.ccsd_contract_workspace_bytes(14, 4, 16, ctypes.byref(n)) == 0     # JACOBI_UPDATE
    assert lib.ccsd_contract_workspace_bytes(15, 4, 16, ctypes.byref(n)) == 1


def test_strassen_levels_are_given_up_where_the_workspace_would_not_fit(lib):
    """ccsd_options.strassen = 1 keeps the workspace within 128 GiB by giving levels up (down to plain products), so that a large
    virtual space never asks for more than plain products + what fits (include/ccsd.h)."""
    from paper_2103_08473_b200.binding import _options
    n = ctypes.c_size_t(0)
    limit = 128 * 2 ** 30
    seen_partial = False
    for shape in ((34, 224, 774), (40, 256, 900), (40, 320, 1080), (20, 364, 1000), (60, 300, 1080)):
        sizes = []
        for mode in (0, 1):
            o = _options(strassen=mode)
            assert lib.ccsd_workspace_bytes(*shape, ctypes.byref(o), ctypes.byref(n)) == 0
            sizes.append(n.value)
        plain, auto = sizes
        assert auto >= plain                                   # levels only ever add operand stacks
        assert auto <= max(limit, plain), (shape, plain, auto)  # and never push the workspace beyond the limit
        seen_partial |= plain < auto < limit and shape != (34, 224, 774)
    assert seen_partial                                        # (40, 256, 900): some levels kept, some given up


def test_strassen_entry_points_validate_on_the_host(lib):
    """ccsd_zgemm_nt_strassen*: size arithmetic and argument checks need no GPU."""
    n = ctypes.c_size_t(0)
    M, N, K = 1031, 97, 1033
    assert lib.ccsd_zgemm_nt_strassen_workspace_bytes(M, N, K, 1, ctypes.byref(n)) == 0
    one = n.value
    mh, nh, kh = (M + 1) // 2, (N + 1) // 2, ((K + 1) // 2 + 1) // 2 * 2
    # two operand stacks (16 B + 8 B plane per element) and seven products, each buffer rounded up to 256 bytes
    assert 7 * (mh * kh + nh * kh) * 24 + 7 * mh * nh * 16 <= one <= 7 * (mh * kh + nh * kh) * 24 + 7 * mh * nh * 16 + 5 * 256
    assert lib.ccsd_zgemm_nt_strassen_workspace_bytes(M, N, K, 2, ctypes.byref(n)) == 0
    assert n.value > one                                                       # 49 quarter-size matrices: 49/16 vs 7/4 of the operand
    for bad in ((0, N, K, 1), (M, 0, K, 1), (M, N, 0, 1), (M, N, K, 0), (M, N, K, 3)):
        assert lib.ccsd_zgemm_nt_strassen_workspace_bytes(*bad, ctypes.byref(n)) == 1
    assert lib.ccsd_zgemm_nt_strassen_workspace_bytes(M, N, K, 1, None) == 1
    buf = ctypes.create_string_buffer(512)
    p = (ctypes.addressof(buf) + 255) // 256 * 256
    call = lambda m, nn, k, a, b, c, lda, ldb, lv, ws, wsb: lib.ccsd_zgemm_nt_strassen(  # noqa: E731
        m, nn, k, a, lda, b, ldb, c, N, 1, 1.0, 0.0, 0, 0, lv, ws, wsb, None)
    assert call(M, N, K, None, p, p, K, K, 1, p, one) == 1                     # null operand
    assert call(M, N, K, p, p, p, K - 1, K, 1, p, one) == 1                    # rows overlap
    assert call(M, N, K, p, p, p, K, K, 3, p, one) == 1                        # levels
    assert call(M, N, K, p, p, p, K, K, 1, p, one - 1) == 1                    # workspace too small
    assert call(M, N, K, p, p, p, K, K, 1, p + 8, one) == 1                    # workspace misaligned
    assert lib.ccsd_strassen_info(None, None) == 4                             # CCSD_ESTATE


def test_null_handles_are_rejected(lib):
    assert lib.ccsd_iterate(None, None, None, None) == 4     # CCSD_ESTATE
    assert lib.ccsd_energy(None, None, None) == 4
    assert lib.ccsd_destroy(None) == 4
    assert lib.ccsd_get_tensor(None, 0, None) == 4


def test_no_cpu_fallback(lib):
    """Without a CUDA device the compute entry points fail loudly instead of computing on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    buf = (ctypes.c_double * 64)()
    p = ctypes.cast(buf, ctypes.c_void_p)
    assert lib.ccsd_zgemm_nt(2, 2, 2, p, 2, p, 2, p, 2, 1, 1.0, 0.0, 0, 0, None) == 3       # CCSD_ECUDA
    ctx = ctypes.c_void_p(None)
    ws = ctypes.c_void_p(256 * 1024)
    assert lib.ccsd_init(ctypes.byref(ctx), p, p, 2, 2, 1, None, ws, 1 << 40, None) == 3
    assert not ctx.value
    n = ctypes.c_size_t(0)
    assert lib.ccsd_zgemm_nt_strassen_workspace_bytes(2, 2, 2, 1, ctypes.byref(n)) == 0
    assert lib.ccsd_zgemm_nt_strassen(2, 2, 2, p, 2, p, 2, p, 2, 1, 1.0, 0.0, 0, 0, 1, ws, n.value, None) == 3
    assert lib.ccsd_energy_static(2, 2, p, p, p, p, p, None) == 3
    import paper_2103_08473_b200 as pkg
    with pytest.raises(RuntimeError):
        pkg.zgemm_nt([[1.0]], [[1.0]])
    import numpy as np
    with pytest.raises(RuntimeError):
        pkg.CCSD(np.eye(4), np.zeros((1, 4, 4)), 2, 2)


def test_product_does_not_import_oracle():
    """The product path shares no code with the oracle and never routes through it."""
    pkg_dir = os.path.join(ROOT, "paper_2103_08473_b200")
    for dirpath, _, files in os.walk(pkg_dir):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.replace("shares nothing with oracle/", "").replace(
                    "no code shared with oracle/", "") or f in ("ccsd_lib.cu", "common.cuh"), f
                assert "import oracle" not in text and "from oracle" not in text, f
    for f in ("ccsd_oracle.py", "ccsd_oracle.c", "cc2_oracle.py", "cc2_oracle.c", "triples_oracle.py", "triples_oracle.c",
              "lambda_oracle.py"):
        text = open(os.path.join(ROOT, "oracle", f)).read()
        assert not re.search(r"^\s*(import|from)\s+paper_2103_08473_b200", text, flags=re.M), f
        assert not re.search(r"#\s*include\s*[<\"].*ccsd\.h", text), f
        assert "csrc" not in text, f


def test_gemm_plan_picks_tiles_against_padding_and_wave_quantisation(lib):
    """ccsd_gemm_plan (host arithmetic): the documented choices of DESIGN.md's kernel section."""
    from paper_2103_08473_b200.binding import gemm_plan
    pe = 16 * 1024 * 1024
    # cfg3: many waves -> padded columns decide.  N = oo = 561 -> 12 x 48; N = nvir = 224 -> 4 x 56; N = nocc = 34 -> 40
    assert gemm_plan(24976, 561, 24976, planes=True, partial_elems=pe) == {"variant": 12, "bm": 128, "bn": 48, "ksplit": 1}
    assert gemm_plan(24976, 224, 816, batch=256, planes=True, partial_elems=pe)["bn"] == 56
    assert gemm_plan(849184, 34, 224, partial_elems=pe)["bn"] == 40
    # cfg2 / cfg1: few waves -> the wave count decides (6 x 100 tiles of 48 columns would be 4.05 waves)
    assert gemm_plan(12720, 276, 12720, planes=True, partial_elems=pe)["bn"] == 56
    assert gemm_plan(4560, 120, 4560, planes=True, partial_elems=pe)["bn"] == 32
    # skinny outputs with a huge K are split deep; without scratch there is no split
    p = gemm_plan(34, 34, 849184, partial_elems=pe)
    assert p["ksplit"] > 100 and gemm_plan(34, 34, 849184)["ksplit"] == 1
    # 4M family on request
    assert gemm_plan(1000, 64, 1000, mode=2)["variant"] in (0, 1, 2, 3, 4)
    assert lib.ccsd_gemm_plan(0, 1, 1, 1, 0, 0, 0, None) == 1
