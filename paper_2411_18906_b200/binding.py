"""Thin ctypes binding over the C ABI of libhea_b200.so (include/hea.h).

Argument marshalling only: every step of the path runs in the CUDA kernels behind the C ABI.  torch is used for
device memory and streams.  There is no CPU fallback: a missing library or a missing device raises.
"""
import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libhea_b200.so")

HEA_OK, HEA_EINVAL, HEA_EUNSUPPORTED, HEA_ENOMEM, HEA_ECUDA = 0, 1, 2, 3, 4
HASH_INIT = 0xCBF29CE484222325
NO_STEP = 0xFFFFFFFFFFFFFFFF
STATS_WORDS = 5            # hea_mc_stats = 4 x uint64 + 1 x double
MOVE_WORDS = 3             # hea_move = uint64 + 3 x uint32 (+ 4 bytes padding)
STATS_DTYPE = np.dtype([("n_accept", "<u8"), ("n_null", "<u8"), ("hash", "<u8"),
                        ("last_accept_step", "<u8"), ("J", "<f8")])
MOVE_DTYPE = np.dtype([("step", "<u8"), ("k", "<u4"), ("a", "<u4"), ("b", "<u4")], align=True)

EXPORTS = ["hea_version", "hea_last_error", "hea_create", "hea_destroy", "hea_info", "hea_neighbor_table",
           "hea_set_option", "hea_get_option", "hea_init_random", "hea_sro_full", "hea_mc_stats_reset",
           "hea_mc_run", "hea_mc_run_ex", "hea_pool_select", "hea_sro_full_host", "hea_mc_run_host", "hea_launch_count", "hea_measure_peaks",
           "hea_pool_rank_static"]


class HeaError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libhea_b200 error {code}: {msg}")
        self.code = code


_lib = None


def lib():
    """Loads the in-tree shared library; raises if it has not been built (python -m paper_2411_18906_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2411_18906_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i32, i64, u64 = C.c_void_p, C.c_int, C.c_int64, C.c_uint64
        L.hea_version.restype = C.c_char_p
        L.hea_last_error.restype = C.c_char_p
        L.hea_create.argtypes = [C.POINTER(vp), i32, i32, i32, i32, i32, vp, i32, vp, vp, i32]
        L.hea_destroy.argtypes = [vp]
        L.hea_info.argtypes = [vp, vp, vp, vp]
        L.hea_neighbor_table.argtypes = [vp, i32, vp]
        L.hea_set_option.argtypes = [vp, C.c_char_p, i64]
        L.hea_get_option.argtypes = [vp, C.c_char_p, vp]
        L.hea_init_random.argtypes = [vp, vp, i64, u64, u64, vp]
        L.hea_sro_full.argtypes = [vp, vp, i64, vp, vp, vp, vp]
        L.hea_mc_stats_reset.argtypes = [vp, vp, i64, vp]
        L.hea_mc_run.argtypes = [vp, vp, vp, i64, u64, i32, u64, u64, u64, vp, vp, i64, vp]
        L.hea_mc_run_ex.argtypes = [vp, vp, vp, i64, u64, i32, u64, u64, u64, vp, vp, i64, i32, u64, vp, vp, vp]
        L.hea_pool_select.argtypes = [vp, vp, vp, vp, i64, i64, u64, u64, vp, vp]
        L.hea_sro_full_host.argtypes = [vp, vp, i64, vp, vp, vp]
        L.hea_mc_run_host.argtypes = [vp, vp, vp, i64, u64, i32, u64, u64, u64, vp]
        L.hea_launch_count.argtypes = [vp, vp]
        L.hea_measure_peaks.argtypes = [vp, vp, i32, vp]
        L.hea_pool_rank_static.argtypes = [vp, vp, i64, i64, vp, vp]
        _lib = L
    return _lib


def _check(rc):
    if rc != HEA_OK:
        raise HeaError(rc, lib().hea_last_error().decode())


def _np(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


class Hea:
    """hea_ctx wrapper.  Same names and arguments as the C calls."""

    def __init__(self, lattice, dims, conc, shell_w, alpha_target, device=0):
        lat = {"fcc": 0, "bcc": 1}[lattice] if isinstance(lattice, str) else int(lattice)
        conc = np.ascontiguousarray(conc, dtype=np.float64)
        shell_w = np.ascontiguousarray(shell_w, dtype=np.float64)
        self.M, self.S = len(conc), len(shell_w)
        t = np.ascontiguousarray(alpha_target, dtype=np.float64)
        if t.size != self.S * self.M * self.M:
            raise ValueError("alpha_target must have S*M*M entries")
        self._h = C.c_void_p()
        _check(lib().hea_create(C.byref(self._h), lat, dims[0], dims[1], dims[2], self.M, _np(conc), self.S,
                                _np(shell_w), _np(t), device))
        self.device = torch.device("cuda", device)
        n = C.c_int64()
        z = np.zeros(3, dtype=np.int32)
        nps = np.zeros(8, dtype=np.int64)
        _check(lib().hea_info(self._h, C.byref(n), _np(z), _np(nps)))
        self.N = int(n.value)
        self.z = [int(v) for v in z[:self.S]]
        self.n_per_species = [int(v) for v in nps[:self.M]]

    def close(self):
        if getattr(self, "_h", None):
            lib().hea_destroy(self._h)
            self._h = None

    __del__ = close

    # ---- setup / introspection
    def neighbor_table(self, shell):
        out = np.zeros((self.N, self.z[shell]), dtype=np.int32)
        _check(lib().hea_neighbor_table(self._h, shell, _np(out)))
        return out

    def set_option(self, name, value):
        _check(lib().hea_set_option(self._h, name.encode(), int(value)))

    def get_option(self, name):
        v = C.c_int64()
        _check(lib().hea_get_option(self._h, name.encode(), C.byref(v)))
        return int(v.value)

    def launch_count(self):
        v = C.c_int64()
        _check(lib().hea_launch_count(self._h, C.byref(v)))
        return int(v.value)

    PEAK_NAMES = ("lds_u8_random_gathers_per_s", "lds_wavefronts_per_s", "alu_pipe_instr_per_s", "fma_pipe_int_instr_per_s",
                  "issue_instr_per_s", "fp64_instr_per_s", "l2_random_sector_GBps", "sm_clock_mhz")

    def measure_peaks(self):
        """hea_measure_peaks: dict of whole-chip rates measured by the library's micro-benchmarks."""
        out = np.zeros(len(self.PEAK_NAMES), dtype=np.float64)
        _check(lib().hea_measure_peaks(self._h, _np(out), len(out), _stream()))
        return dict(zip(self.PEAK_NAMES, (float(v) for v in out)))

    # ---- device-buffer calls (torch tensors own the memory; asynchronous on the current stream)
    def init_random(self, n_chains, seed, chain0=0, out=None):
        occ = out if out is not None else torch.empty((n_chains, self.N), dtype=torch.uint8, device=self.device)
        _check(lib().hea_init_random(self._h, C.c_void_p(occ.data_ptr()), n_chains, seed, chain0, _stream()))
        return occ

    def sro_full(self, occ, want_alpha=True, want_obj=True, counts=None):
        assert occ.dtype == torch.uint8 and occ.is_cuda and occ.is_contiguous() and occ.shape[-1] == self.N
        B = occ.numel() // self.N
        if counts is None:
            counts = torch.empty((B, self.S, self.M, self.M), dtype=torch.int32, device=self.device)
        alpha = torch.empty((B, self.S, self.M, self.M), dtype=torch.float64, device=self.device) if want_alpha else None
        obj = torch.empty((B,), dtype=torch.float64, device=self.device) if want_obj else None
        _check(lib().hea_sro_full(self._h, C.c_void_p(occ.data_ptr()), B, C.c_void_p(counts.data_ptr()),
                                  C.c_void_p(alpha.data_ptr()) if want_alpha else None,
                                  C.c_void_p(obj.data_ptr()) if want_obj else None, _stream()))
        return counts, alpha, obj

    def new_stats(self, n_chains):
        st = torch.empty((n_chains, STATS_WORDS), dtype=torch.int64, device=self.device)
        _check(lib().hea_mc_stats_reset(self._h, C.c_void_p(st.data_ptr()), n_chains, _stream()))
        return st

    def reset_stats(self, stats):
        _check(lib().hea_mc_stats_reset(self._h, C.c_void_p(stats.data_ptr()), stats.shape[0], _stream()))
        return stats

    def mc_run(self, occ, counts, n_steps, K, seed, chain0=0, step0=0, stats=None, log_cap=0):
        """In place on occ [C][N] and counts [C][S][M][M]; returns (stats tensor [C][5] int64 view, log or None)."""
        assert occ.dtype == torch.uint8 and occ.is_cuda and occ.is_contiguous() and occ.dim() == 2
        assert counts.dtype == torch.int32 and counts.is_cuda and counts.is_contiguous()
        n = occ.shape[0]
        if stats is None:
            stats = self.new_stats(n)
        log = torch.zeros((n, max(log_cap, 1), MOVE_WORDS), dtype=torch.int64, device=self.device) if log_cap > 0 else None
        _check(lib().hea_mc_run(self._h, C.c_void_p(occ.data_ptr()), C.c_void_p(counts.data_ptr()), n, n_steps, K,
                                seed, chain0, step0, C.c_void_p(stats.data_ptr()),
                                C.c_void_p(log.data_ptr()) if log is not None else None, log_cap, _stream()))
        return stats, log

    def mc_run_ex(self, occ, counts, n_steps, K, seed, chain0=0, step0=0, stats=None, log_cap=0, select_best=False,
                  depth_limit=0, depth=None):
        """hea_mc_run_ex: best-of-K selection and search-depth termination.  Returns (stats, log, depth, steps_done)."""
        n = occ.shape[0]
        if stats is None:
            stats = self.new_stats(n)
        if depth is None:
            depth = torch.zeros((n,), dtype=torch.int64, device=self.device)
        steps_done = torch.zeros((n,), dtype=torch.int64, device=self.device)
        log = torch.zeros((n, max(log_cap, 1), MOVE_WORDS), dtype=torch.int64, device=self.device) if log_cap > 0 else None
        _check(lib().hea_mc_run_ex(self._h, C.c_void_p(occ.data_ptr()), C.c_void_p(counts.data_ptr()), n, n_steps, K,
                                   seed, chain0, step0, C.c_void_p(stats.data_ptr()),
                                   C.c_void_p(log.data_ptr()) if log is not None else None, log_cap,
                                   1 if select_best else 0, depth_limit, C.c_void_p(depth.data_ptr()),
                                   C.c_void_p(steps_done.data_ptr()), _stream()))
        return stats, log, depth, steps_done

    def pool_select(self, occ, counts, stats, n_keep, seed, new_chain0):
        """hea_pool_select, in place; returns order [n_keep] int32 (previous index of each kept chain)."""
        n = occ.shape[0]
        order = torch.empty((max(n_keep, 1),), dtype=torch.int32, device=self.device)
        _check(lib().hea_pool_select(self._h, C.c_void_p(occ.data_ptr()), C.c_void_p(counts.data_ptr()),
                                     C.c_void_p(stats.data_ptr()), n, n_keep, seed, new_chain0,
                                     C.c_void_p(order.data_ptr()), _stream()))
        return order[:n_keep]

    POOL_RANK_STATIC_MAX = 65536

    def pool_rank_static(self, counts, n_keep, order):
        """hea_pool_rank_static: order[:n_keep] = chain indices by ascending J; allocates nothing (order is the caller's)."""
        _check(lib().hea_pool_rank_static(self._h, C.c_void_p(counts.data_ptr()), counts.shape[0], n_keep,
                                          C.c_void_p(order.data_ptr()), _stream()))
        return order[:n_keep]

    # ---- host-buffer (end-to-end) calls: numpy arrays in, synchronous
    def sro_full_host(self, occ, want_alpha=False, want_obj=True):
        occ = np.ascontiguousarray(occ, dtype=np.uint8).reshape(-1, self.N)
        B = occ.shape[0]
        counts = np.empty((B, self.S, self.M, self.M), dtype=np.int32)
        alpha = np.empty((B, self.S, self.M, self.M), dtype=np.float64) if want_alpha else None
        obj = np.empty((B,), dtype=np.float64) if want_obj else None
        _check(lib().hea_sro_full_host(self._h, _np(occ), B, _np(counts), _np(alpha), _np(obj)))
        return counts, alpha, obj

    def mc_run_host(self, occ, n_steps, K, seed, chain0=0, step0=0, stats=None, counts_out=None):
        """occ: numpy [C][N] uint8, updated in place.  Returns (counts, stats) numpy arrays."""
        assert occ.dtype == np.uint8 and occ.flags.c_contiguous and occ.ndim == 2 and occ.shape[1] == self.N
        n = occ.shape[0]
        if stats is None:
            stats = fresh_stats_host(n)
        counts = counts_out if counts_out is not None else np.empty((n, self.S, self.M, self.M), dtype=np.int32)
        _check(lib().hea_mc_run_host(self._h, _np(occ), _np(counts), n, n_steps, K, seed, chain0, step0, _np(stats)))
        return counts, stats


def fresh_stats_host(n):
    st = np.zeros(n, dtype=STATS_DTYPE)
    st["hash"] = HASH_INIT
    st["last_accept_step"] = NO_STEP
    return st


def stats_to_numpy(stats_tensor):
    """[C][5] int64 device tensor -> structured numpy array (J reinterpreted as float64)."""
    raw = stats_tensor.cpu().numpy()
    return np.ascontiguousarray(raw).view(STATS_DTYPE).reshape(-1)


def log_to_numpy(log_tensor):
    raw = np.ascontiguousarray(log_tensor.cpu().numpy())
    return raw.view(MOVE_DTYPE).reshape(raw.shape[0], raw.shape[1])
