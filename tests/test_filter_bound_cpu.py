"""CPU check of the reject filter's error bound, with no GPU and no kernel code.

The filter of mc_halo_kernel drops a candidate when an fp32 quadratic form of the first-shell count differences F exceeds
a per-(p, q) threshold T' = roundup_fp32(max(1.001 J_cur, floor) - C~ + E).  This test restates the table build and the
fp32 evaluation in numpy exactly as DESIGN.md 6.3 states them, and checks against EXACT rational arithmetic
(fractions.Fraction over the fp64 inputs) that
  (Lemma 1)  |fp32 value - exact value of the form| <= the E the table build computes, for random admissible F, and that
             a dropped candidate has an exact first-shell term X' >= theta;
  (Lemma 2)  a candidate whose exact first-shell term is >= theta is not improving for the oracle's fp64 objective
             (one shell, so that J is the first-shell term itself: the tightest case).
It is a test of the derivation, independent of the CUDA code; the GPU-side counterpart aims real candidates at the
threshold (tests/test_gpu_round2.py::test_reject_filter_at_the_accept_threshold)."""
from fractions import Fraction as Fr

import numpy as np
import pytest

from oracle import hea_oracle as ho
from paper_2411_18906_b200 import workloads as wl

F32 = np.float32


def fma32(a, b, c):
    # a * b is exact in fp64 for fp32 inputs; one rounding to fp64 of the sum precedes the rounding to fp32 (a double
    # rounding that differs from a true fma by at most one fp32 ulp in rare cases: far inside the bound under test)
    return F32(np.float64(a) * np.float64(b) + np.float64(c))


def roundup32(x):
    f = F32(x)
    return f if Fr(float(f)) >= Fr(float(x)) else np.nextafter(f, F32(np.inf))


def build_table(N1, g, t, w1, J_cur, z1, floor):
    """Row (p, q) of the filter table as DESIGN.md 6.3 / the "reject filter" block of hea_mc2.cu build it (fp64 arithmetic,
    coefficients rounded to fp32, threshold rounded up).  N1, g, t: [M][M] of the first shell."""
    M = N1.shape[0]
    nstar = (1.0 - t) / g
    W = (w1 * g) * g
    be = N1.astype(np.float64) - nstar
    eb = 4.44e-16 * (np.abs(nstar) + np.abs(be))
    Cq = float((W * be * be).sum())
    EC = float((W * (2.0 * np.abs(be) + eb) * eb).sum())
    b2 = 2.0 * be
    e2 = 2.0 * eb
    Fm = 2.0 * z1
    rows = {}
    for p in range(M):
        for q in range(M):
            if p == q:
                continue
            L = np.zeros(M, dtype=F32); Q = np.zeros(M, dtype=F32); c = np.zeros(M, dtype=F32)
            A = B = 0.0
            for r in range(M):
                if r == p:
                    t1, t2, Qr, cr = 2.0 * W[p, p] * b2[p, p], -2.0 * W[p, q] * b2[p, q], 4.0 * W[p, p], -1.0
                    et = 2.0 * W[p, p] * e2[p, p] + 2.0 * W[p, q] * e2[p, q]
                elif r == q:
                    t1, t2, Qr, cr = -2.0 * W[q, q] * b2[q, q], 2.0 * W[p, q] * b2[p, q], 4.0 * W[q, q], 1.0
                    et = 2.0 * W[q, q] * e2[q, q] + 2.0 * W[p, q] * e2[p, q]
                else:
                    t1, t2, Qr, cr = 2.0 * W[p, r] * b2[p, r], -2.0 * W[q, r] * b2[q, r], 2.0 * (W[p, r] + W[q, r]), 0.0
                    et = 2.0 * W[p, r] * e2[p, r] + 2.0 * W[q, r] * e2[q, r]
                L[r], Q[r], c[r] = F32(t1 + t2), F32(Qr), F32(cr)
                A += (abs(t1) + abs(t2)) * Fm + Qr * Fm * Fm
                B += et * Fm
            X = 2.0 * W[p, q]
            A += X * 4.0 * Fm * Fm
            E = 1.9073486328125e-6 * A + 1.000001 * (B + EC) + 1.0e-12 * abs(Cq)
            theta = max(1.001 * J_cur, floor)
            rows[(p, q)] = dict(L=L, Q=Q, c=c, X=F32(X), T=roundup32(theta - Cq + E), E=E, Cq=Cq, theta=theta)
    return rows


def eval32(row, F):
    acc, D = F32(0.0), F32(0.0)
    for r in range(len(F)):
        f = F32(F[r])
        acc = fma32(fma32(row["Q"][r], f, row["L"][r]), f, acc)
        D = fma32(row["c"][r], f, D)
    return fma32(F32(row["X"] * D), D, acc)


def exact_terms(N1, g, t, w1, p, q, F):
    """(C, X') in exact rational arithmetic on the fp64 inputs."""
    M = N1.shape[0]
    C = X = Fr(0)
    for i in range(M):
        for j in range(M):
            gi, ti = Fr(float(g[i, j])), Fr(float(t[i, j]))
            W = Fr(float(w1)) * gi * gi
            beta = Fr(int(N1[i, j])) - (1 - ti) / gi
            ci, cj = int(i == p) - int(i == q), int(j == p) - int(j == q)
            dN = ci * int(F[j]) + cj * int(F[i])
            C += W * beta * beta
            X += W * (beta + dN) ** 2
    return C, X


def contexts():
    out = []
    # (name, workload, MC steps before the table is taken: far from / near the optimum)
    w1 = wl.Workload(name="a", lattice="fcc", dims=(6, 6, 6), conc=[0.25] * 4, n_shells=1, shell_w=[1.0], n_chains=1, n_steps=0,
                     K=32, seed=3, target_seed=11, target_range=(-0.2, 0.2))
    w2 = wl.Workload(name="b", lattice="bcc", dims=(8, 8, 8), conc=[0.2] * 5, n_shells=1, shell_w=[0.7], n_chains=1, n_steps=0,
                     K=32, seed=4, target_seed=7, target_range=(-0.15, 0.15))
    w3 = wl.Workload(name="c", lattice="fcc", dims=(5, 5, 5), conc=[0.4, 0.4, 0.1, 0.1], n_shells=1, shell_w=[1.0], n_chains=1,
                     n_steps=0, K=32, seed=5, target_seed=13, target_range=(-0.1, 0.1))
    for w in (w1, w2, w3):
        for steps in (0, 300, 20000):
            out.append((w, steps))
    return out


@pytest.mark.parametrize("w,steps", contexts())
def test_filter_bound_and_decisions(w, steps):
    o = ho.Oracle(*w.create_args())
    occ = o.init_random(1, w.seed)
    cnt = np.stack([o.pair_counts(occ[0])])
    if steps:
        o.mc_run(occ, cnt, steps, w.K, w.seed, eval_all=False)
    M, z1 = o.M, o.z[0]
    N1 = cnt[0, 0].astype(np.int64)
    Nsp = np.array(o.n_per_species, dtype=np.float64)
    g = np.array([[float(o.N) / float(z1 * Nsp[i] * Nsp[j]) for j in range(M)] for i in range(M)])
    t = o.target[0]
    w1 = float(o.shell_w[0])
    J_cur = o.objective(cnt[0])
    inv_c_max = max(np.sqrt(o.N * z1 * g[i, i]) for i in range(M))
    Amax = 2.0 * inv_c_max + 2.0 + np.abs(t).max()
    floor = 1.0e-18 * w1 * max(1.0, (Amax / 100.0) ** 2)
    rows = build_table(N1, g, t, w1, J_cur, z1, floor)
    rs = np.random.RandomState(steps + M)
    n_drop = n_keep = 0
    for trial in range(400):
        p, q = (int(v) for v in rs.choice(M, 2, replace=False))
        F = rs.randint(-z1, z1 + 1, size=M)
        if trial % 3 == 0:
            F = rs.randint(-2, 3, size=M)                       # the small differences of a converged chain
        F[-1] -= F.sum()                                        # the differences of a shell sum to zero
        if abs(F[-1]) > 2 * z1:
            continue
        row = rows[(p, q)]
        lt = eval32(row, F)
        C, X = exact_terms(N1, g, t, w1, p, q, F)
        l_exact = X - C
        # Lemma 1: the fp32 value is within E of the exact form (E also absorbs |C~ - C|)
        assert abs(Fr(float(lt)) - l_exact) + abs(Fr(row["Cq"]) - C) <= Fr(row["E"])
        dropped = bool(lt > row["T"])
        if dropped:
            n_drop += 1
            assert X >= Fr(row["theta"])                        # ... hence a dropped candidate has X' >= theta
            # Lemma 2 (one shell: J' is the first-shell term): the oracle's fp64 objective does not improve
            cnt2 = cnt[0].copy()
            for i in range(M):
                for j in range(M):
                    cnt2[0, i, j] += (int(i == p) - int(i == q)) * int(F[j]) + (int(j == p) - int(j == q)) * int(F[i])
            assert not (o.objective(cnt2) < J_cur)
        else:
            n_keep += 1
    assert n_drop > 50                                          # the filter does drop (it is not vacuous) ...
    for (p, q), row in rows.items():                            # ... and never the candidate that changes nothing (l = 0 <= T')
        assert not (eval32(row, np.zeros(M, dtype=np.int64)) > row["T"])


def test_filter_threshold_is_rounded_up():
    for x in (1e-10, 3.3333333e-7, 1.0 + 2 ** -30, 5e-20, 1e-46):
        f = roundup32(x)
        assert Fr(float(f)) >= Fr(x)
        assert float(np.nextafter(f, F32(-np.inf))) < x or float(f) == x
