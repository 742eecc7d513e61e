"""ctypes binding of include/ccsd.h (argument marshalling only; same names as the C entry points)."""
from __future__ import annotations

import contextlib
import ctypes
import os

HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None

STATUS = {0: "CCSD_OK", 1: "CCSD_EINVAL", 2: "CCSD_ENOMEM", 3: "CCSD_ECUDA", 4: "CCSD_ESTATE", 5: "CCSD_ESINGULAR",
          6: "CCSD_ENOTCONVERGED"}
TENSOR_IDS = {"fock": 0, "vvvv": 1, "vovv": 2, "vovo": 3, "oovv": 4, "ooov": 5, "oooo": 6, "tau": 10, "Hvv": 11,
              "Gvv": 12, "Hoo": 13, "Goo": 14, "Hov": 15, "Hvovo": 16, "C": 17, "A": 18, "S1": 19, "S2": 20,
              "S2_ring": 30, "S2_goo": 31, "S2_vdag_t1": 32, "S2_gvv": 33, "S2_c_t1": 34, "S2_hh_ladder": 35,
              "S2_pp_ladder": 36, "S2_driver": 37}
TERM_IDS = {"pp_ladder": 0, "hh_ladder": 1, "ring": 2, "tau": 3, "pp_ladder_planes": 4,
            "f_ov": 5, "f_vv": 6, "f_oo": 7, "w_oooo": 8, "w_ovvo": 9, "c_ovoo": 10,
            "s1_residual": 11, "s2_small_terms": 12, "energy": 13, "jacobi_update": 14}
NSTEPS = 16

# every symbol include/ccsd.h declares
EXPORTS = ["ccsd_default_options", "ccsd_workspace_bytes", "ccsd_init", "ccsd_iterate", "ccsd_energy", "ccsd_residual",
           "ccsd_get_amplitudes", "ccsd_set_amplitudes", "ccsd_tensor_elems", "ccsd_get_tensor", "ccsd_destroy",
           "ccsd_contract_workspace_bytes", "ccsd_contract", "ccsd_zgemm_nt", "ccsd_zgemm_nt_planes", "ccsd_sum_plane", "ccsd_transpose",
           "ccsd_enable_step_timing", "ccsd_get_step_times", "ccsd_get_init_stats", "ccsd_step_name", "ccsd_launch_count",
           "ccsd_measure_fp64_peak", "ccsd_real_flops_per_cmac", "ccsd_strerror",
           "ccsd_last_cuda_error", "ccsd_triples_workspace_bytes", "ccsd_triples", "ccsd_get_triples_times",
           "ccsd_triples_block", "ccsd_triples_count", "ccsd_triples_range", "ccsd_t1_diagnostic", "ccsd_solve", "ccsd_lambda_workspace_bytes",
           "ccsd_lambda_init", "ccsd_lambda_iterate", "ccsd_lambda_solve", "ccsd_lambda_residual", "ccsd_get_lambda", "ccsd_set_lambda",
           "ccsd_get_lambda_residual", "ccsd_density", "ccsd_expectation", "ccsd_update", "ccsd_shard_info",
           "ccsd_shard_ranges", "ccsd_gemm_plan", "ccsd_energy_static",
           "ccsd_zgemm_nt_strassen_workspace_bytes", "ccsd_zgemm_nt_strassen", "ccsd_strassen_info"]

# limits of ccsd_energy_static (include/ccsd.h): its scratch is a fixed device array inside the library
ENERGY_STATIC_MAX_NOCC = 128
ENERGY_STATIC_MAX_NVIR = 512
ENERGY_STATIC_SCRATCH_BYTES = 1121024


class CCSDError(RuntimeError):
    def __init__(self, status: int, where: str):
        lib = load_library()
        msg = lib.ccsd_strerror(status).decode()
        cuda = lib.ccsd_last_cuda_error().decode()
        super().__init__(f"{where}: {STATUS.get(status, status)} ({msg}){' [' + cuda + ']' if cuda else ''}")
        self.status = status


class Options(ctypes.Structure):
    _fields_ = [("ndiis", ctypes.c_int), ("level_shift", ctypes.c_double), ("gemm_mode", ctypes.c_int),
                ("ccd", ctypes.c_int), ("cc2", ctypes.c_int), ("direct_ladder", ctypes.c_int), ("graph", ctypes.c_int),
                ("shard_rank", ctypes.c_int), ("shard_world", ctypes.c_int), ("strassen", ctypes.c_int)]


def lib_path() -> str:
    return os.path.join(HERE, "libccsd_b200.so")


def load_library():
    """dlopen the in-tree CUDA library; fails loudly if it has not been built (no fallback)."""
    global _LIB
    if _LIB is None:
        path = lib_path()
        if not os.path.exists(path):
            # a fresh checkout has no built artefact (*.so is git-ignored): compile it once, in-tree, if nvcc is there
            try:
                from . import build as _build
                _build.build()
            except Exception as exc:                                   # noqa: BLE001
                raise ImportError(f"{path} is missing and could not be built ({exc}): run "
                                  "`python -m paper_2103_08473_b200.build` (needs nvcc); there is no CPU fallback")
        lib = ctypes.CDLL(path)
        vp, i64, dbl = ctypes.c_void_p, ctypes.c_int64, ctypes.c_double
        lib.ccsd_default_options.argtypes = [ctypes.POINTER(Options)]
        lib.ccsd_default_options.restype = None
        lib.ccsd_workspace_bytes.argtypes = [ctypes.c_int] * 3 + [ctypes.POINTER(Options), ctypes.POINTER(ctypes.c_size_t)]
        lib.ccsd_init.argtypes = [ctypes.POINTER(vp), vp, vp, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                  ctypes.POINTER(Options), vp, ctypes.c_size_t, vp]
        lib.ccsd_iterate.argtypes = [vp] + [ctypes.POINTER(dbl)] * 3
        lib.ccsd_energy.argtypes = [vp] + [ctypes.POINTER(dbl)] * 2
        lib.ccsd_residual.argtypes = [vp]
        lib.ccsd_update.argtypes = [vp] + [ctypes.POINTER(dbl)] * 3
        lib.ccsd_shard_info.argtypes = [vp, ctypes.POINTER(i64)]
        lib.ccsd_shard_ranges.argtypes = [ctypes.c_int] * 4 + [ctypes.POINTER(i64)]
        lib.ccsd_gemm_plan.argtypes = [i64, i64, i64, i64, ctypes.c_int, ctypes.c_int, i64, ctypes.POINTER(ctypes.c_int)]
        lib.ccsd_lambda_workspace_bytes.argtypes = [vp, ctypes.POINTER(ctypes.c_size_t)]
        lib.ccsd_lambda_init.argtypes = [vp, vp, ctypes.c_size_t]
        lib.ccsd_lambda_iterate.argtypes = [vp, ctypes.POINTER(dbl)]
        lib.ccsd_lambda_solve.argtypes = [vp, ctypes.c_double, ctypes.c_int, ctypes.POINTER(ctypes.c_int), ctypes.POINTER(dbl)]
        lib.ccsd_lambda_residual.argtypes = [vp]
        lib.ccsd_get_lambda.argtypes = [vp, vp, vp]
        lib.ccsd_set_lambda.argtypes = [vp, vp, vp, ctypes.c_int]
        lib.ccsd_get_lambda_residual.argtypes = [vp, vp, vp]
        lib.ccsd_density.argtypes = [vp, vp]
        lib.ccsd_expectation.argtypes = [vp, vp, vp, ctypes.POINTER(dbl), ctypes.POINTER(dbl)]
        lib.ccsd_solve.argtypes = [vp, dbl, ctypes.c_int, ctypes.POINTER(ctypes.c_int)] + [ctypes.POINTER(dbl)] * 3
        lib.ccsd_t1_diagnostic.argtypes = [vp, ctypes.POINTER(dbl)]
        lib.ccsd_get_amplitudes.argtypes = [vp, vp, vp]
        lib.ccsd_set_amplitudes.argtypes = [vp, vp, vp, ctypes.c_int]
        lib.ccsd_tensor_elems.argtypes = [vp, ctypes.c_int, ctypes.POINTER(ctypes.c_size_t)]
        lib.ccsd_get_tensor.argtypes = [vp, ctypes.c_int, vp]
        lib.ccsd_destroy.argtypes = [vp]
        lib.ccsd_contract_workspace_bytes.argtypes = [ctypes.c_int] * 3 + [ctypes.POINTER(ctypes.c_size_t)]
        lib.ccsd_contract.argtypes = [ctypes.c_int] * 3 + [ctypes.POINTER(vp), vp, ctypes.c_int,
                                                            ctypes.POINTER(Options), vp, ctypes.c_size_t, vp]
        lib.ccsd_energy_static.argtypes = [ctypes.c_int, ctypes.c_int, vp, vp, vp, vp, vp, vp]
        lib.ccsd_zgemm_nt.argtypes = [i64, i64, i64, vp, i64, vp, i64, vp, i64, i64, dbl, dbl, ctypes.c_int,
                                      ctypes.c_int, vp]
        lib.ccsd_zgemm_nt_strassen_workspace_bytes.argtypes = [i64, i64, i64, ctypes.c_int, ctypes.POINTER(ctypes.c_size_t)]
        lib.ccsd_zgemm_nt_strassen.argtypes = [i64, i64, i64, vp, i64, vp, i64, vp, i64, i64, dbl, dbl, ctypes.c_int,
                                               ctypes.c_int, ctypes.c_int, vp, ctypes.c_size_t, vp]
        lib.ccsd_strassen_info.argtypes = [vp, ctypes.POINTER(ctypes.c_int)]
        lib.ccsd_sum_plane.argtypes = [vp, vp, i64, vp]
        lib.ccsd_zgemm_nt_planes.argtypes = [i64, i64, i64, vp, i64, vp, vp, i64, vp, vp, i64, i64, dbl, dbl, ctypes.c_int,
                                             ctypes.c_int, vp]
        lib.ccsd_transpose.argtypes = [vp, vp, ctypes.POINTER(i64), ctypes.POINTER(ctypes.c_int), ctypes.c_int, vp]
        lib.ccsd_enable_step_timing.argtypes = [vp, ctypes.c_int]
        lib.ccsd_get_step_times.argtypes = [vp, ctypes.POINTER(ctypes.c_float)]
        lib.ccsd_get_init_stats.argtypes = [vp, ctypes.POINTER(dbl)]
        lib.ccsd_step_name.argtypes = [ctypes.c_int]
        lib.ccsd_step_name.restype = ctypes.c_char_p
        lib.ccsd_launch_count.argtypes = [ctypes.c_int]
        lib.ccsd_launch_count.restype = ctypes.c_longlong
        lib.ccsd_measure_fp64_peak.argtypes = [ctypes.POINTER(dbl), vp, ctypes.c_int, vp]
        lib.ccsd_real_flops_per_cmac.argtypes = [ctypes.POINTER(Options)]
        lib.ccsd_strerror.argtypes = [ctypes.c_int]
        lib.ccsd_strerror.restype = ctypes.c_char_p
        lib.ccsd_last_cuda_error.restype = ctypes.c_char_p
        lib.ccsd_triples_workspace_bytes.argtypes = [vp, ctypes.POINTER(ctypes.c_size_t)]
        lib.ccsd_triples.argtypes = [vp] + [ctypes.POINTER(dbl)] * 3 + [vp, ctypes.c_size_t]
        lib.ccsd_get_triples_times.argtypes = [vp, ctypes.POINTER(ctypes.c_float)]
        lib.ccsd_triples_count.argtypes = [vp, ctypes.POINTER(ctypes.c_int64)]
        lib.ccsd_triples_range.argtypes = [vp, ctypes.c_int64, ctypes.c_int64] + [ctypes.POINTER(dbl)] * 3 + [vp, ctypes.c_size_t]
        lib.ccsd_triples_block.argtypes = [vp, ctypes.c_int, ctypes.c_int, ctypes.c_int, vp, vp, vp, vp, ctypes.c_size_t]
        _LIB = lib
    return _LIB


def _step_names():
    lib = load_library()
    return [lib.ccsd_step_name(k).decode() for k in range(NSTEPS)]


class _LazyNames(list):
    def _fill(self):
        if not len(self):
            self.extend(_step_names())

    def __iter__(self):
        self._fill()
        return super().__iter__()

    def __getitem__(self, k):
        self._fill()
        return super().__getitem__(k)


STEP_NAMES = _LazyNames()


def _check(status: int, where: str):
    if status != 0:
        raise CCSDError(status, where)


def _workspace(torch, nbytes: int):
    """A device workspace of nbytes (+ alignment slack).  The large ones (tens of GB) get a segment of their own: torch's
    caching allocator would otherwise carve them out of a bigger cached segment (say the 115 GiB one a previous solver
    left), whose remainder can then neither serve the next large request nor go back to the driver while this one lives."""
    if nbytes >= (4 << 30):
        torch.cuda.empty_cache()
    try:
        return torch.empty(int(nbytes) + 256, dtype=torch.uint8, device="cuda")
    except torch.OutOfMemoryError:
        torch.cuda.empty_cache()
        return torch.empty(int(nbytes) + 256, dtype=torch.uint8, device="cuda")


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2103_08473_b200 needs a CUDA device (B200); there is no CPU fallback")
    return torch


def _stream_ptr(torch):
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def _dev_c128(torch, x):
    """host numpy / torch tensor -> contiguous complex128 CUDA tensor (marshalling only)."""
    if not isinstance(x, torch.Tensor):
        x = torch.from_numpy(x)
    return x.to(device="cuda", dtype=torch.complex128).contiguous()


def shard_ranges(nocc: int, nvir: int, rank: int, world: int) -> dict:
    """ccsd_shard_ranges (host arithmetic only): the slab of rank `rank` of `world`."""
    arr = (ctypes.c_int64 * 8)()
    _check(load_library().ccsd_shard_ranges(int(nocc), int(nvir), int(rank), int(world), arr), "ccsd_shard_ranges")
    return dict(zip(("a_lo", "a_hi", "w_lo", "w_hi", "ij_lo", "ij_hi", "wa_lo", "wa_hi"), (int(x) for x in arr)))


def gemm_plan(M: int, N: int, K: int, batch: int = 1, mode: int = 0, planes: bool = False, partial_elems: int = 0) -> dict:
    """ccsd_gemm_plan (host arithmetic only): tile variant and split-K depth the DMMA GEMM would use for this shape."""
    arr = (ctypes.c_int * 4)()
    _check(load_library().ccsd_gemm_plan(int(M), int(N), int(K), int(batch), int(mode), int(bool(planes)), int(partial_elems), arr),
           "ccsd_gemm_plan")
    return {"variant": arr[0], "bm": arr[1], "bn": arr[2], "ksplit": arr[3]}


def launch_count(reset: bool = False) -> int:
    return int(load_library().ccsd_launch_count(1 if reset else 0))


def real_flops_per_cmac(gemm_mode: int = 0) -> int:
    """8 (4M) or 6 (3M): real flops the DMMA GEMMs execute per complex multiply-add (ccsd_real_flops_per_cmac)."""
    opts = _options(gemm_mode=gemm_mode)
    return int(load_library().ccsd_real_flops_per_cmac(ctypes.byref(opts)))


def measure_fp64_peak(launches: int = 10) -> float:
    """DMMA.8x8x4 issue-rate yardstick in TFLOP/s (ccsd_measure_fp64_peak)."""
    torch = _torch()
    lib = load_library()
    scratch = torch.zeros(8, dtype=torch.float64, device="cuda")
    out = ctypes.c_double(0.0)
    _check(lib.ccsd_measure_fp64_peak(ctypes.byref(out), scratch.data_ptr(), int(launches), _stream_ptr(torch)),
           "ccsd_measure_fp64_peak")
    return float(out.value)


def _options(ndiis=6, level_shift=0.0, gemm_mode=0, ccd=False, cc2=False, direct_ladder=False, graph=True,
             shard=(0, 1), strassen=1) -> Options:
    return Options(int(ndiis), float(level_shift), int(gemm_mode), int(bool(ccd)), int(bool(cc2)), int(bool(direct_ladder)),
                   int(graph), int(shard[0]), int(shard[1]), int(strassen))


class CCSD:
    """ccsd_init / ccsd_iterate / ccsd_energy / ccsd_get_* on device tensors.

    h [n][n] and B [naux][n][n] may be numpy arrays (copied host->device here) or CUDA complex128 tensors.
    Every context works on ONE stream, `self.stream`: the caller's current stream at construction, unless that is the
    default stream -- CUDA graphs cannot be captured there -- in which case the context gets a torch stream of its own
    (pass `stream=` to choose).  Methods may be called from any current stream: every library call is bracketed by
    device-side stream waits (_on_stream), tensors are allocated on the caller's stream.
    """

    def __init__(self, h, B, nocc: int, nvir: int, ndiis: int = 6, level_shift: float = 0.0, gemm_mode: int = 0,
                 ccd: bool = False, cc2: bool = False, direct_ladder: bool = False, graph: int = 1, stream=None,
                 shard=None, group=None, strassen: int = 1):
        torch = _torch()
        lib = load_library()
        self._lib, self._torch = lib, torch
        if stream is None:
            stream = torch.cuda.current_stream()
            if stream.cuda_stream == torch.cuda.default_stream().cuda_stream:
                stream = torch.cuda.Stream()
        self.stream = stream
        self._ctx = ctypes.c_void_p(None)
        # shard = (rank, world): this context evaluates rank's slab of the iteration (ccsd_options.shard_rank / shard_world);
        # iterate() then sums the packed S2 over `group` (torch.distributed; None = the default group) between ccsd_residual
        # and ccsd_update.  shard=None: one GPU does everything.
        self.shard = (0, 1) if shard is None else (int(shard[0]), int(shard[1]))
        self.group = group
        opts = _options(ndiis, level_shift, gemm_mode, ccd, cc2, direct_ladder, graph, self.shard, strassen)
        self.nocc, self.nvir, self.n = int(nocc), int(nvir), int(nocc + nvir)
        self.oo = self.nocc * (self.nocc - 1) // 2
        self.vv = self.nvir * (self.nvir - 1) // 2
        self.naux = int(B.shape[0])
        assert tuple(h.shape) == (self.n, self.n) and tuple(B.shape) == (self.naux, self.n, self.n)
        self._opts = opts
        nbytes = ctypes.c_size_t(0)
        _check(lib.ccsd_workspace_bytes(self.nocc, self.nvir, self.naux, ctypes.byref(self._opts),
                                        ctypes.byref(nbytes)), "ccsd_workspace_bytes")
        self.workspace_bytes = int(nbytes.value)
        self._lam_ws = None
        # the workspace first: the (much smaller) device copies of h and B would otherwise be carved out of whatever large
        # cached segment a previous solver left and pin it while the workspace is allocated (see _workspace)
        self._ws = _workspace(torch, self.workspace_bytes)
        h_d, B_d = _dev_c128(torch, h), _dev_c128(torch, B)
        base = (self._ws.data_ptr() + 255) // 256 * 256
        self._ctx = ctypes.c_void_p(None)
        with self._on_stream():
            _check(lib.ccsd_init(ctypes.byref(self._ctx), h_d.data_ptr(), B_d.data_ptr(), self.nocc, self.nvir, self.naux,
                                 ctypes.byref(self._opts), base, self.workspace_bytes,
                                 ctypes.c_void_p(self.stream.cuda_stream)), "ccsd_init")

    @contextlib.contextmanager
    def _on_stream(self):
        """Bracket library calls: the context's stream first waits for the caller's current stream (inputs made there are
        ready); afterwards the caller's stream waits for it (results are ready for whatever the caller enqueues next).
        Device-side ordering only."""
        torch = self._torch
        caller = torch.cuda.current_stream()
        if caller.cuda_stream == self.stream.cuda_stream:
            yield
            return
        self.stream.wait_stream(caller)
        try:
            yield
        finally:
            caller.wait_stream(self.stream)

    def _call(self, fn, *args, where=None, ok=(0,)):
        with self._on_stream():
            st = fn(self._ctx, *args)
        if st not in ok:
            _check(st, where or fn.__name__)
        return st

    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx.value:
            self.stream.synchronize()                 # nothing of this context is in flight when its memory goes back
            self._lib.ccsd_destroy(self._ctx)
            self._ctx = ctypes.c_void_p(None)
            self._ws = None
            self._lam_ws = None
            self._trip_ws = None
            if self.workspace_bytes >= (4 << 30):     # hand tens of GB back to the driver rather than to torch's cache
                self._torch.cuda.empty_cache()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def shard_info(self) -> dict:
        arr = (ctypes.c_int64 * 12)()
        self._call(self._lib.ccsd_shard_info, arr, where="ccsd_shard_info")
        keys = ("rank", "world", "a_lo", "a_hi", "w_lo", "w_hi", "ij_lo", "ij_hi", "s2_offset", "s2_elems", "s1_offset", "s1_elems")
        return dict(zip(keys, (int(x) for x in arr)))

    def s2_view(self):
        """The context's S2 buffer [(i<j)][(a<b)] as a torch view of the workspace (no copy): what the all-reduce of a sharded
        iteration acts on."""
        torch = self._torch
        info = self.shard_info()
        off = info["s2_offset"] + ((self._ws.data_ptr() + 255) // 256 * 256 - self._ws.data_ptr())
        return self._ws[off:off + info["s2_elems"] * 16].view(torch.complex128).view(self.oo, self.vv)

    def update(self):
        """ccsd_update: Jacobi + DIIS + energy from the residuals the context holds -> (E_corr, ||S/D||_2)."""
        er, ei, sn = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
        self._call(self._lib.ccsd_update, ctypes.byref(er), ctypes.byref(ei), ctypes.byref(sn), where="ccsd_update", ok=(0, 5))
        return complex(er.value, ei.value), sn.value

    def iterate(self):
        """One CCSD iteration -> (complex E_corr of the new amplitudes, ||S/D||_2).  In a sharded context: this rank's slab
        of the residual, ONE all-reduce of the packed S2 over the group (on the context's stream), the replicated update."""
        if self.shard[1] > 1:
            from .sharding import allreduce_complex_
            self.residual()
            s2 = self.s2_view()
            with self._on_stream(), self._torch.cuda.stream(self.stream):
                allreduce_complex_(s2, self.group)
            return self.update()
        er, ei, sn = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
        self._call(self._lib.ccsd_iterate, ctypes.byref(er), ctypes.byref(ei), ctypes.byref(sn), where="ccsd_iterate", ok=(0, 5))
        return complex(er.value, ei.value), sn.value

    def energy(self) -> complex:
        er, ei = ctypes.c_double(), ctypes.c_double()
        self._call(self._lib.ccsd_energy, ctypes.byref(er), ctypes.byref(ei), where="ccsd_energy")
        return complex(er.value, ei.value)

    def solve(self, tol: float = 1e-9, max_iterations: int = 30):
        """ccsd_solve -> (converged, iterations, complex E_corr, ||S/D||_2); defaults = the paper's .TCONVERG / .NCYCLES."""
        it, er, ei, sn = ctypes.c_int(), ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
        st = self._call(self._lib.ccsd_solve, float(tol), int(max_iterations), ctypes.byref(it), ctypes.byref(er),
                        ctypes.byref(ei), ctypes.byref(sn), where="ccsd_solve", ok=(0, 6))
        return st == 0, it.value, complex(er.value, ei.value), sn.value

    def t1_diagnostic(self) -> float:
        out = ctypes.c_double()
        self._call(self._lib.ccsd_t1_diagnostic, ctypes.byref(out), where="ccsd_t1_diagnostic")
        return out.value

    def residual(self):
        self._call(self._lib.ccsd_residual, where="ccsd_residual")

    def get_amplitudes(self):
        torch = self._torch
        t1 = torch.empty((self.nocc, self.nvir), dtype=torch.complex128, device="cuda")
        t2p = torch.empty((self.oo, self.vv), dtype=torch.complex128, device="cuda")
        self._call(self._lib.ccsd_get_amplitudes, t1.data_ptr(), t2p.data_ptr(), where="ccsd_get_amplitudes")
        return t1, t2p

    def set_amplitudes(self, t1, t2p, reset_diis: bool = True):
        torch = self._torch
        t1_d, t2_d = _dev_c128(torch, t1), _dev_c128(torch, t2p)
        assert tuple(t1_d.shape) == (self.nocc, self.nvir) and tuple(t2_d.shape) == (self.oo, self.vv)
        self._call(self._lib.ccsd_set_amplitudes, t1_d.data_ptr(), t2_d.data_ptr(), int(reset_diis), where="ccsd_set_amplitudes")
        self.stream.synchronize()

    def get_tensor(self, name: str):
        torch = self._torch
        tid = TENSOR_IDS[name]
        ne = ctypes.c_size_t(0)
        self._call(self._lib.ccsd_tensor_elems, tid, ctypes.byref(ne), where="ccsd_tensor_elems")
        out = torch.empty(int(ne.value), dtype=torch.complex128, device="cuda")
        self._call(self._lib.ccsd_get_tensor, tid, out.data_ptr(), where=f"ccsd_get_tensor({name})")
        return out

    def _triples_workspace(self):
        """The triples workspace, allocated on first use and kept until close() (a fresh multi-GiB cudaMalloc per call costs
        tenths of a second beside a 5 s computation)."""
        if getattr(self, "_trip_ws", None) is None:
            nbytes = ctypes.c_size_t(0)
            self._call(self._lib.ccsd_triples_workspace_bytes, ctypes.byref(nbytes), where="ccsd_triples_workspace_bytes")
            self._trip_ws = (_workspace(self._torch, nbytes.value), int(nbytes.value))
        ws, nbytes = self._trip_ws
        return ws, (ws.data_ptr() + 255) // 256 * 256, nbytes

    def triples(self) -> dict:
        """+T / (T) / -T corrections at the current amplitudes (ccsd_triples): {"+T": E, "(T)": E, "-T": E} (complex)."""
        ws, base, nbytes = self._triples_workspace()
        a, b, c = (ctypes.c_double * 2)(), (ctypes.c_double * 2)(), (ctypes.c_double * 2)()
        self._call(self._lib.ccsd_triples, a, b, c, base, nbytes, where="ccsd_triples")
        del ws
        return {"+T": complex(a[0], a[1]), "(T)": complex(b[0], b[1]), "-T": complex(c[0], c[1])}

    def triples_count(self) -> int:
        n = ctypes.c_int64(0)
        self._call(self._lib.ccsd_triples_count, ctypes.byref(n), where="ccsd_triples_count")
        return int(n.value)

    def triples_range(self, first: int, count: int) -> dict:
        """Partial sums of +T / (T) / -T over the occupied triples first .. first+count-1 (ccsd_triples_range)."""
        ws, base, nbytes = self._triples_workspace()
        a, b, c = (ctypes.c_double * 2)(), (ctypes.c_double * 2)(), (ctypes.c_double * 2)()
        self._call(self._lib.ccsd_triples_range, int(first), int(count), a, b, c, base, nbytes, where="ccsd_triples_range")
        del ws
        return {"+T": complex(a[0], a[1]), "(T)": complex(b[0], b[1]), "-T": complex(c[0], c[1])}

    def triples_sharded(self, group=None) -> dict:
        """The triples corrections shared among the ranks of a torch.distributed group (every rank holds the same
        amplitudes): each rank evaluates its contiguous range of the occupied triples i<j<k, the six doubles are summed
        with one all-reduce (NCCL: on the device).  Without an initialised process group this is triples()."""
        import torch.distributed as dist
        from .sharding import shard_range, allreduce_energies
        if not (dist.is_available() and dist.is_initialized()):
            return self.triples()
        rank, world = dist.get_rank(group), dist.get_world_size(group)
        first, count = shard_range(self.triples_count(), rank, world)
        return allreduce_energies(self.triples_range(first, count), group=group, device="cuda")

    def triples_times(self) -> dict:
        arr = (ctypes.c_float * 2)()
        self._call(self._lib.ccsd_get_triples_times, arr, where="ccsd_get_triples_times")
        return {"w_gemm_ms": float(arr[0]), "energy_ms": float(arr[1])}

    def triples_block(self, i: int, j: int, k: int):
        """Dense Wbar, Zbar, Ybar [a][b][c] of one occupied triple i<j<k (ccsd_triples_block)."""
        torch = self._torch
        ws, base, nbytes = self._triples_workspace()
        v = self.nvir
        out = [torch.empty((v, v, v), dtype=torch.complex128, device="cuda") for _ in range(3)]
        self._call(self._lib.ccsd_triples_block, int(i), int(j), int(k), out[0].data_ptr(), out[1].data_ptr(), out[2].data_ptr(), base, nbytes, where="ccsd_triples_block")
        self.stream.synchronize()
        del ws
        return out

    # ---- Lambda equations / density (Appendix 7.4-7.5) ----
    def lambda_init(self):
        torch = self._torch
        nbytes = ctypes.c_size_t(0)
        self._call(self._lib.ccsd_lambda_workspace_bytes, ctypes.byref(nbytes), where="ccsd_lambda_workspace_bytes")
        self._lam_ws = None                                # a previous Lambda workspace is released first
        self._lam_ws = _workspace(torch, nbytes.value)    # lives with the solver
        base = (self._lam_ws.data_ptr() + 255) // 256 * 256
        self._call(self._lib.ccsd_lambda_init, base, int(nbytes.value), where="ccsd_lambda_init")

    def lambda_iterate(self) -> float:
        sn = ctypes.c_double()
        self._call(self._lib.ccsd_lambda_iterate, ctypes.byref(sn), where="ccsd_lambda_iterate", ok=(0, 5))
        return sn.value

    def lambda_solve(self, tol: float = 1e-9, max_iterations: int = 30):
        """ccsd_lambda_solve -> (converged, iterations, ||R/D||_2)."""
        it, sn = ctypes.c_int(), ctypes.c_double()
        st = self._call(self._lib.ccsd_lambda_solve, float(tol), int(max_iterations), ctypes.byref(it), ctypes.byref(sn),
                        where="ccsd_lambda_solve", ok=(0, 6))
        return st == 0, it.value, sn.value

    def lambda_residual(self):
        torch = self._torch
        self._call(self._lib.ccsd_lambda_residual, where="ccsd_lambda_residual")
        r1 = torch.empty((self.nocc, self.nvir), dtype=torch.complex128, device="cuda")
        r2p = torch.empty((self.oo, self.vv), dtype=torch.complex128, device="cuda")
        self._call(self._lib.ccsd_get_lambda_residual, r1.data_ptr(), r2p.data_ptr(), where="ccsd_get_lambda_residual")
        self.stream.synchronize()
        return r1, r2p

    def get_lambda(self):
        torch = self._torch
        l1 = torch.empty((self.nocc, self.nvir), dtype=torch.complex128, device="cuda")
        l2p = torch.empty((self.oo, self.vv), dtype=torch.complex128, device="cuda")
        self._call(self._lib.ccsd_get_lambda, l1.data_ptr(), l2p.data_ptr(), where="ccsd_get_lambda")
        self.stream.synchronize()
        return l1, l2p

    def set_lambda(self, l1, l2p, reset_diis: bool = True):
        torch = self._torch
        a, b = _dev_c128(torch, l1), _dev_c128(torch, l2p)
        assert tuple(a.shape) == (self.nocc, self.nvir) and tuple(b.shape) == (self.oo, self.vv)
        self._call(self._lib.ccsd_set_lambda, a.data_ptr(), b.data_ptr(), int(reset_diis), where="ccsd_set_lambda")
        self.stream.synchronize()

    def density(self):
        torch = self._torch
        D = torch.empty((self.n, self.n), dtype=torch.complex128, device="cuda")
        self._call(self._lib.ccsd_density, D.data_ptr(), where="ccsd_density")
        self.stream.synchronize()
        return D

    def expectation(self, D, O) -> complex:
        """eq 16: sum_pq O[p][q] D[p][q] (ccsd_expectation); D from density(), O any [n][n] operator matrix."""
        torch = self._torch
        D_d, O_d = _dev_c128(torch, D), _dev_c128(torch, O)
        assert tuple(D_d.shape) == (self.n, self.n) and tuple(O_d.shape) == (self.n, self.n)
        re, im = ctypes.c_double(), ctypes.c_double()
        self._call(self._lib.ccsd_expectation, D_d.data_ptr(), O_d.data_ptr(), ctypes.byref(re), ctypes.byref(im), where="ccsd_expectation")
        return complex(re.value, im.value)

    def strassen_steps(self) -> dict:
        """{name of a timed step (step_times()): Strassen levels L of its product}; such a product executes (7/8)^L of the
        plain product's flops."""
        info = (ctypes.c_int * 4)()
        self._call(self._lib.ccsd_strassen_info, info, where="ccsd_strassen_info")
        out = {}
        if info[1]:
            out["Hvovo_quad"] = out["ring_gemm"] = int(info[1])
        if info[2]:
            out["pp_ladder"] = int(info[2])
        if info[3]:
            out["C_ovoo"] = int(info[3])
        return out

    def enable_step_timing(self, enable: bool = True):
        self._call(self._lib.ccsd_enable_step_timing, int(enable), where="ccsd_enable_step_timing")

    def init_stats(self) -> dict:
        """How ccsd_init built the packed <ab||cd> (ccsd_get_init_stats): device ms and elements moved."""
        arr = (ctypes.c_double * 5)()
        self._call(self._lib.ccsd_get_init_stats, arr, where="ccsd_get_init_stats")
        return {"gemm_ms": arr[0], "transpose_ms": arr[1], "pack_ms": arr[2], "transposed_elems": arr[3], "packed_elems": arr[4]}

    def step_times(self):
        arr = (ctypes.c_float * NSTEPS)()
        self._call(self._lib.ccsd_get_step_times, arr, where="ccsd_get_step_times")
        return {n: float(arr[k]) for k, n in enumerate(STEP_NAMES)}


def contract(term: str, nocc: int, nvir: int, inputs, out=None, accumulate: bool = False, gemm_mode: int = 0,
             level_shift: float = 0.0, ccd: bool = False):
    """ccsd_contract on CUDA tensors; returns out ([(i<j)][(a<b)] for the ladder/ring/tau terms, the layouts of
    include/ccsd.h for the intermediates f_ov ... c_ovoo and for s1_residual, s2_small_terms, energy (one element) and
    jacobi_update (u1 followed by packed u2; level_shift and ccd apply to it only))."""
    torch = _torch()
    lib = load_library()
    tid = TERM_IDS[term]
    oo, vv = nocc * (nocc - 1) // 2, nvir * (nvir - 1) // 2
    # the sum planes of "pp_ladder_planes" (inputs[2:]) are real float64 CUDA tensors made by sum_plane()
    ins = [_dev_c128(torch, x) for x in inputs[:2]] + list(inputs[2:])
    if tid >= TERM_IDS["f_ov"]:   # the intermediates of eqs 24-31: every input complex128, output shape per term
        ins = [_dev_c128(torch, x) for x in inputs]
        shape = {"f_ov": (nocc, nvir), "f_vv": (nvir, nvir), "f_oo": (nocc, nocc), "w_oooo": (oo, oo),
                 "w_ovvo": (nvir, nocc, nvir, nocc), "c_ovoo": (nocc, nvir, oo),
                 "s1_residual": (nocc, nvir), "s2_small_terms": (oo, vv), "energy": (1,),
                 "jacobi_update": (nocc * nvir + oo * vv,)}[term]
        if out is None:
            out = torch.zeros(shape, dtype=torch.complex128, device="cuda")
    if out is None:
        out = torch.zeros((oo, vv), dtype=torch.complex128, device="cuda")
    nbytes = ctypes.c_size_t(0)
    _check(lib.ccsd_contract_workspace_bytes(tid, nocc, nvir, ctypes.byref(nbytes)), "ccsd_contract_workspace_bytes")
    ws = _workspace(torch, nbytes.value)
    base = (ws.data_ptr() + 255) // 256 * 256
    arr = (ctypes.c_void_p * len(ins))(*[x.data_ptr() for x in ins])
    opts = _options(gemm_mode=gemm_mode, level_shift=level_shift, ccd=ccd)
    _check(lib.ccsd_contract(tid, nocc, nvir, arr, out.data_ptr(), int(accumulate), ctypes.byref(opts), base,
                             int(nbytes.value), _stream_ptr(torch)), f"ccsd_contract({term})")
    torch.cuda.current_stream().synchronize()   # ws / ins must outlive the enqueued kernels
    return out


def energy_static(nocc: int, nvir: int, f, oovv, t1, t2p, out):
    """ccsd_energy_static: the correlation energy (eq 9) of the amplitudes (t1, t2p) without any workspace -- the library's
    fixed device scratch is used (nocc <= ENERGY_STATIC_MAX_NOCC, nvir <= ENERGY_STATIC_MAX_NVIR, CCSDError beyond).  Nothing is
    allocated or copied here either: every argument must already be a contiguous complex128 CUDA tensor (f [n][n],
    oovv [(k<l)][(c<d)], t1 [i][a], t2p [(i<j)][(a<b)], out one element, overwritten).  Asynchronous on the current stream;
    calls that overlap on the GPU race on the shared scratch (include/ccsd.h).  Returns out."""
    torch = _torch()
    lib = load_library()
    oo, vv = nocc * (nocc - 1) // 2, nvir * (nvir - 1) // 2
    for name, x, elems in (("f", f, (nocc + nvir) ** 2), ("oovv", oovv, oo * vv), ("t1", t1, nocc * nvir),
                           ("t2p", t2p, oo * vv), ("out", out, 1)):
        if not (isinstance(x, torch.Tensor) and x.is_cuda and x.dtype == torch.complex128 and x.is_contiguous()
                and x.numel() == elems):
            raise ValueError(f"energy_static: {name} must be a contiguous complex128 CUDA tensor of {elems} elements")
    _check(lib.ccsd_energy_static(nocc, nvir, f.data_ptr(), oovv.data_ptr(), t1.data_ptr(), t2p.data_ptr(), out.data_ptr(),
                                  _stream_ptr(torch)), "ccsd_energy_static")
    return out


def zgemm_nt(A, B, C=None, alpha: complex = 1.0, accumulate: bool = False, mode: int = 0, transposed_out: bool = False,
             planes=None):
    """C[m][n] (+)= alpha * sum_k A[m][k] B[n][k]; transposed_out stores C as [n][m].
    planes = (As, Bs): float64 CUDA sum planes of A and B (sum_plane()) -> ccsd_zgemm_nt_planes."""
    torch = _torch()
    lib = load_library()
    A, B = _dev_c128(torch, A), _dev_c128(torch, B)
    M, K = A.shape
    N = B.shape[0]
    assert B.shape[1] == K
    if C is None:
        C = torch.zeros((N, M) if transposed_out else (M, N), dtype=torch.complex128, device="cuda")
    csm, csn = (1, M) if transposed_out else (N, 1)
    alpha = complex(alpha)
    if planes is not None:
        As, Bs = planes
        assert As.shape == A.shape and Bs.shape == B.shape and As.dtype == torch.float64 and Bs.dtype == torch.float64
        _check(lib.ccsd_zgemm_nt_planes(M, N, K, A.data_ptr(), K, As.data_ptr(), B.data_ptr(), K, Bs.data_ptr(),
                                        C.data_ptr(), csm, csn, alpha.real, alpha.imag, int(accumulate), mode,
                                        _stream_ptr(torch)), "ccsd_zgemm_nt_planes")
        torch.cuda.current_stream().synchronize()
        return C
    _check(lib.ccsd_zgemm_nt(M, N, K, A.data_ptr(), K, B.data_ptr(), K, C.data_ptr(), csm, csn, alpha.real, alpha.imag,
                             int(accumulate), mode, _stream_ptr(torch)), "ccsd_zgemm_nt")
    torch.cuda.current_stream().synchronize()
    return C


def zgemm_nt_strassen(A, B, C=None, alpha: complex = 1.0, accumulate: bool = False, mode: int = 0, transposed_out: bool = False,
                      levels: int = 1, sync: bool = True):
    """zgemm_nt by one or two Strassen levels (ccsd_zgemm_nt_strassen): 7 half-size / 49 quarter-size products in one batched
    DMMA launch.  sync=False returns (C, workspace) without waiting (timing loops: keep the workspace alive)."""
    torch = _torch()
    lib = load_library()
    A, B = _dev_c128(torch, A), _dev_c128(torch, B)
    M, K = A.shape
    N = B.shape[0]
    assert B.shape[1] == K
    if C is None:
        C = torch.zeros((N, M) if transposed_out else (M, N), dtype=torch.complex128, device="cuda")
    csm, csn = (1, M) if transposed_out else (N, 1)
    alpha = complex(alpha)
    nbytes = ctypes.c_size_t(0)
    _check(lib.ccsd_zgemm_nt_strassen_workspace_bytes(M, N, K, levels, ctypes.byref(nbytes)), "ccsd_zgemm_nt_strassen_workspace_bytes")
    ws = _workspace(torch, nbytes.value)
    base = (ws.data_ptr() + 255) // 256 * 256
    _check(lib.ccsd_zgemm_nt_strassen(M, N, K, A.data_ptr(), K, B.data_ptr(), K, C.data_ptr(), csm, csn, alpha.real, alpha.imag,
                                      int(accumulate), mode, levels, base, int(nbytes.value), _stream_ptr(torch)),
           "ccsd_zgemm_nt_strassen")
    if not sync:
        return C, ws
    torch.cuda.current_stream().synchronize()   # ws must outlive the enqueued kernels
    return C


def sum_plane(x):
    """3M operand sum plane Re x + Im x of a complex128 CUDA tensor (ccsd_sum_plane); same shape, float64."""
    torch = _torch()
    lib = load_library()
    x = _dev_c128(torch, x)
    out = torch.empty(x.shape, dtype=torch.float64, device="cuda")
    _check(lib.ccsd_sum_plane(x.data_ptr(), out.data_ptr(), x.numel(), _stream_ptr(torch)), "ccsd_sum_plane")
    return out


def transpose(x, perm, conj: bool = False):
    """4-index transposition out[...perm...] = x (ccsd_transpose); x is a 4-d CUDA complex128 tensor."""
    torch = _torch()
    lib = load_library()
    x = _dev_c128(torch, x)
    assert x.dim() == 4 and sorted(perm) == [0, 1, 2, 3]
    dims = (ctypes.c_int64 * 4)(*x.shape)
    pr = (ctypes.c_int * 4)(*perm)
    out = torch.empty([x.shape[p] for p in perm], dtype=torch.complex128, device="cuda")
    _check(lib.ccsd_transpose(x.data_ptr(), out.data_ptr(), dims, pr, int(conj), _stream_ptr(torch)), "ccsd_transpose")
    return out
