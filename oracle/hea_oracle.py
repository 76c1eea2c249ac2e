"""ctypes loader for the CPU ORACLE (oracle/hea_oracle.c).

TEST INFRASTRUCTURE ONLY: import from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs.  Nothing under paper_2411_18906_b200/ may import this module, and this module
imports nothing from that package.  Argument marshalling only; all arithmetic is in the C file.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hea_oracle.c")
_LIB = os.path.join(_HERE, "libhea_oracle.so")
CFLAGS = ["-O2", "-ffp-contract=off", "-std=c11", "-Wall", "-shared", "-fPIC", "-pthread"]

HASH0 = 0xCBF29CE484222325
NO_STEP = 0xFFFFFFFFFFFFFFFF
STATS_DTYPE = np.dtype([("n_accept", "<u8"), ("n_null", "<u8"), ("hash", "<u8"),
                        ("last_accept_step", "<u8"), ("J", "<f8")])
MOVE_DTYPE = np.dtype([("step", "<u8"), ("k", "<u4"), ("a", "<u4"), ("b", "<u4")], align=True)


def build(force=False):
    """Compile the oracle with gcc (never -ffast-math; no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", *CFLAGS, _SRC, "-o", _LIB, "-lm"])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        vp, i32, i64, u32, u64 = C.c_void_p, C.c_int, C.c_int64, C.c_uint32, C.c_uint64
        L.ora_create.restype = vp
        L.ora_create.argtypes = [i32, i32, i32, i32, i32, vp, i32, vp, vp]
        L.ora_destroy.argtypes = [vp]
        L.ora_info.argtypes = [vp, vp, vp, vp]
        L.ora_neighbor_table.argtypes = [vp, i32, vp]
        L.ora_philox4x32_10.argtypes = [vp, vp, vp]
        L.ora_init_random.argtypes = [vp, vp, i64, u64, u64]
        L.ora_pair_counts.argtypes = [vp, vp, vp]
        L.ora_alpha.argtypes = [vp, vp, vp]
        L.ora_objective.restype = C.c_double
        L.ora_objective.argtypes = [vp, vp]
        L.ora_sro_full.argtypes = [vp, vp, i64, vp, vp, vp]
        L.ora_sro_full_mt.restype = i32
        L.ora_sro_full_mt.argtypes = [vp, vp, i64, vp, vp, vp, i32]
        L.ora_propose.restype = i32
        L.ora_propose.argtypes = [vp, vp, u64, u64, u64, u32, vp, vp]
        L.ora_delta_counts.argtypes = [vp, vp, u32, u32, vp]
        L.ora_mc_run.restype = i32
        L.ora_mc_run.argtypes = [vp, vp, vp, i64, u64, i32, u64, u64, u64, vp, vp, i64, i32, i32]
        L.ora_mc_run_ex.restype = i32
        L.ora_mc_run_ex.argtypes = [vp, vp, vp, i64, u64, i32, u64, u64, u64, vp, vp, i64, i32, u64, vp, vp]
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().ora_philox4x32_10(_p(c), _p(k), _p(out))
    return out


def fresh_stats(n):
    st = np.zeros(n, dtype=STATS_DTYPE)
    st["hash"] = HASH0
    st["last_accept_step"] = NO_STEP
    return st


class Oracle:
    """One lattice + composition + target (the arguments of hea_create)."""

    def __init__(self, lattice, dims, conc, shell_w, alpha_target):
        lat = {"fcc": 0, "bcc": 1}[lattice] if isinstance(lattice, str) else int(lattice)
        conc = np.ascontiguousarray(conc, dtype=np.float64)
        shell_w = np.ascontiguousarray(shell_w, dtype=np.float64)
        self.M, self.S = len(conc), len(shell_w)
        t = np.ascontiguousarray(alpha_target, dtype=np.float64).reshape(self.S, self.M, self.M)
        self._h = lib().ora_create(lat, dims[0], dims[1], dims[2], self.M, _p(conc), self.S, _p(shell_w), _p(t))
        if not self._h:
            raise ValueError("ora_create rejected the arguments")
        n = C.c_int64()
        z = np.zeros(3, dtype=np.int32)
        nps = np.zeros(8, dtype=np.int64)
        lib().ora_info(self._h, C.byref(n), _p(z), _p(nps))
        self.N = int(n.value)
        self.z = [int(v) for v in z[:self.S]]
        self.n_per_species = [int(v) for v in nps[:self.M]]
        self.conc, self.shell_w, self.target = conc, shell_w, t

    def __del__(self):
        if getattr(self, "_h", None):
            lib().ora_destroy(self._h)
            self._h = None

    def neighbor_table(self, shell):
        out = np.zeros((self.N, self.z[shell]), dtype=np.int32)
        lib().ora_neighbor_table(self._h, shell, _p(out))
        return out

    def init_random(self, n_chains, seed, chain0=0):
        occ = np.zeros((n_chains, self.N), dtype=np.uint8)
        lib().ora_init_random(self._h, _p(occ), n_chains, seed, chain0)
        return occ

    def pair_counts(self, occ):
        occ = np.ascontiguousarray(occ, dtype=np.uint8)
        assert occ.shape == (self.N,)
        counts = np.zeros((self.S, self.M, self.M), dtype=np.int32)
        lib().ora_pair_counts(self._h, _p(occ), _p(counts))
        return counts

    def alpha(self, counts):
        counts = np.ascontiguousarray(counts, dtype=np.int32).reshape(self.S, self.M, self.M)
        out = np.zeros((self.S, self.M, self.M), dtype=np.float64)
        lib().ora_alpha(self._h, _p(counts), _p(out))
        return out

    def objective(self, counts):
        counts = np.ascontiguousarray(counts, dtype=np.int32).reshape(self.S, self.M, self.M)
        return float(lib().ora_objective(self._h, _p(counts)))

    def sro_full(self, occ, n_threads=1):
        occ = np.ascontiguousarray(occ, dtype=np.uint8).reshape(-1, self.N)
        B = occ.shape[0]
        counts = np.zeros((B, self.S, self.M, self.M), dtype=np.int32)
        alpha = np.zeros((B, self.S, self.M, self.M), dtype=np.float64)
        J = np.zeros(B, dtype=np.float64)
        used = lib().ora_sro_full_mt(self._h, _p(occ), B, _p(counts), _p(alpha), _p(J), n_threads)
        self.threads_used = used
        return counts, alpha, J

    def propose(self, occ, seed, chain, step, k):
        a, b = C.c_uint32(), C.c_uint32()
        ok = lib().ora_propose(self._h, _p(occ), seed, chain, step, k, C.byref(a), C.byref(b))
        return bool(ok), int(a.value), int(b.value)

    def delta_counts(self, occ, a, b, counts):
        """Returns counts + the pair-count change of exchanging sites a and b (occ is the state before)."""
        out = np.ascontiguousarray(counts, dtype=np.int32).copy()
        lib().ora_delta_counts(self._h, _p(occ), a, b, _p(out))
        return out

    def mc_run(self, occ, counts, n_steps, K, seed, chain0=0, step0=0, stats=None, log_cap=0,
               n_threads=1, eval_all=True):
        """In-place on occ [C][N] and counts [C][S][M][M]; returns (stats, log)."""
        assert occ.dtype == np.uint8 and occ.flags.c_contiguous and occ.ndim == 2 and occ.shape[1] == self.N
        assert counts.dtype == np.int32 and counts.flags.c_contiguous
        n = occ.shape[0]
        if stats is None:
            stats = fresh_stats(n)
        log = np.zeros((n, log_cap), dtype=MOVE_DTYPE) if log_cap > 0 else None
        used = lib().ora_mc_run(self._h, _p(occ), _p(counts), n, n_steps, K, seed, chain0, step0, _p(stats),
                                _p(log), log_cap, n_threads, 1 if eval_all else 0)
        self.threads_used = used
        return stats, log

    def pool_select(self, occ, counts, stats, n_keep, seed, new_chain0):
        """SURVEY 8f-2, the selection step of the global search (Alg. 1; the retained top
        solutions seed the next iteration, the others are generated entirely randomly).  Reading (A24):
        the pool is ranked by J of the supplied counts, ascending, ties -> lower index; the n_keep best move to the front
        in rank order with their counts and stats; every other slot r >= n_keep gets a fresh seeded random configuration
        (D8, chain id new_chain0 + r - n_keep), its recount, and reset stats.  In place; returns `order`, the previous
        index of the chain now at each kept position.  Plain numpy over the pinned pieces (objective, init, recount)."""
        n = occ.shape[0]
        J = np.array([self.objective(counts[c]) for c in range(n)])
        order = sorted(range(n), key=lambda c: (J[c], c))[:n_keep]
        occ[:n_keep], counts[:n_keep], stats[:n_keep] = occ[order].copy(), counts[order].copy(), stats[order].copy()
        if n > n_keep:
            occ[n_keep:] = self.init_random(n - n_keep, seed, new_chain0)
            for c in range(n_keep, n):
                counts[c] = self.pair_counts(occ[c])
            stats[n_keep:] = fresh_stats(n - n_keep)
        return np.asarray(order, dtype=np.int32)

    def mc_run_ex(self, occ, counts, n_steps, K, seed, chain0=0, step0=0, stats=None, log_cap=0, select_best=False,
                  depth_limit=0, depth=None):
        """SURVEY 8f-1 options: best-of-K selection, search-depth termination.  Returns (stats, log, depth, steps_done)."""
        n = occ.shape[0]
        if stats is None:
            stats = fresh_stats(n)
        if depth is None:
            depth = np.zeros(n, dtype=np.uint64)
        steps_done = np.zeros(n, dtype=np.uint64)
        log = np.zeros((n, log_cap), dtype=MOVE_DTYPE) if log_cap > 0 else None
        lib().ora_mc_run_ex(self._h, _p(occ), _p(counts), n, n_steps, K, seed, chain0, step0, _p(stats), _p(log),
                            log_cap, 1 if select_best else 0, depth_limit, _p(depth), _p(steps_done))
        return stats, log, depth, steps_done
