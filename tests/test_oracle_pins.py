"""Pins for the CPU oracle (oracle/hea_oracle.c) against things other than itself:
published known-answer vectors, O(N^2) geometry, closed forms for ordered structures, sum rules, exact
expectations, brute-force enumeration.  CPU only (-m "not gpu").  Citations: DESIGN.md section 3 (D1-D9),
PAPER.md Eq. 2-4, SURVEY.md section 8(c)."""
import itertools
import math
import os

import numpy as np
import pytest

from oracle import hea_oracle as ho
from paper_2411_18906_b200 import workloads as wl

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def make(lattice, dims, conc, S, w=None, target=None):
    M = len(conc)
    w = [1.0, 0.5, 0.25][:S] if w is None else w
    t = np.zeros((S, M, M)) if target is None else target
    return ho.Oracle(lattice, dims, conc, w, t)


# ------------------------------------------------------------------ D7: Philox known answers
def test_philox_known_answer_vectors():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        assert ho.philox4x32_10(v[0:4], v[4:6]).tolist() == v[6:10]


def test_workload_target_generator_uses_same_philox():
    # the input generator's private Philox (word 0 only) agrees with the pinned one
    for ctr, key in [((0, 0, 0, 0), (0, 0)), ((5, 0, 0xFFFFFFFE, 0), (7, 0)), ((0xFFFFFFFF,) * 4, (0xFFFFFFFF,) * 2)]:
        assert wl._philox_word0(ctr, key) == int(ho.philox4x32_10(ctr, key)[0])


# ------------------------------------------------------------------ D1-D2: lattice + table
def positions(lattice, dims):
    """Independent restatement of D1: doubled integer coordinates of every site, in site order."""
    basis = {"fcc": [(0, 0, 0), (0, 1, 1), (1, 0, 1), (1, 1, 0)], "bcc": [(0, 0, 0), (1, 1, 1)]}[lattice]
    out = []
    for x in range(dims[0]):
        for y in range(dims[1]):
            for z in range(dims[2]):
                for b in basis:
                    out.append((2 * x + b[0], 2 * y + b[1], 2 * z + b[2]))
    return np.array(out, dtype=np.int64)


SHELL_D2 = {"fcc": [2, 4, 6], "bcc": [3, 4, 8]}
SHELL_Z = {"fcc": [12, 6, 24], "bcc": [8, 6, 12]}


@pytest.mark.parametrize("lattice,dims", [("fcc", (3, 3, 3)), ("fcc", (3, 4, 5)), ("bcc", (3, 3, 3)),
                                          ("bcc", (4, 3, 5)), ("fcc", (5, 5, 5)), ("bcc", (6, 6, 6))])
def test_table_equals_minimum_image_distance_search(lattice, dims):
    o = make(lattice, dims, [0.5, 0.5] if (np.prod(dims) * (4 if lattice == "fcc" else 2)) % 2 == 0 else [1.0], 3)
    assert o.z == SHELL_Z[lattice]
    pos = positions(lattice, dims)
    assert len(pos) == o.N
    box = 2 * np.array(dims)
    d = pos[:, None, :] - pos[None, :, :]
    d = (d + box // 2) % box - box // 2          # minimum image (box sides are even; L >= 3 so shells are unambiguous)
    d2 = (d ** 2).sum(-1)
    for s in range(3):
        tab = o.neighbor_table(s)
        assert tab.shape == (o.N, SHELL_Z[lattice][s])
        for a in range(o.N):
            want = np.nonzero(d2[a] == SHELL_D2[lattice][s])[0]
            assert len(want) == SHELL_Z[lattice][s]
            assert sorted(tab[a].tolist()) == want.tolist()          # distinct neighbours, exactly the shell


@pytest.mark.parametrize("lattice,dims", [("fcc", (1, 1, 1)), ("fcc", (2, 2, 2)), ("bcc", (1, 2, 3)),
                                          ("bcc", (2, 2, 2)), ("fcc", (2, 3, 1)), ("fcc", (4, 4, 4))])
def test_table_symmetric_with_multiplicity_and_distinctness_thresholds(lattice, dims):
    N = (4 if lattice == "fcc" else 2) * int(np.prod(dims))
    o = make(lattice, dims, [0.5, 0.5], 3)
    for s in range(3):
        tab = o.neighbor_table(s)
        mult = np.zeros((N, N), dtype=np.int64)
        for a in range(N):
            for v in tab[a]:
                mult[a, v] += 1
        assert (mult == mult.T).all()
        assert (mult.sum(1) == SHELL_Z[lattice][s]).all()
        distinct = (mult <= 1).all() and (np.diag(mult) == 0).all()
        need = 2 if s == 0 else 3
        if min(dims) >= need:
            assert distinct


def test_offsets_are_lexicographically_ordered():
    # entry k of site 0 is the site at offset o_k; recover o_k from positions (L large enough to be unambiguous)
    for lattice in ("fcc", "bcc"):
        dims = (5, 5, 5)
        o = make(lattice, dims, [1.0], 3)
        pos = positions(lattice, dims)
        box = 2 * np.array(dims)
        for s in range(3):
            tab = o.neighbor_table(s)
            for a in (0, 7, o.N - 1):
                offs = [tuple(((pos[v] - pos[a] + box // 2) % box - box // 2).tolist()) for v in tab[a]]
                assert offs == sorted(offs)
                assert all(sum(c * c for c in off) == SHELL_D2[lattice][s] for off in offs)


# ------------------------------------------------------------------ D3: species counts
def test_species_counts():
    assert make("fcc", (5, 5, 5), [0.4, 0.4, 0.1, 0.1], 1).n_per_species == [200, 200, 50, 50]
    assert make("bcc", (2, 2, 2), [1 / 3, 1 / 3, 1 / 3], 1).n_per_species == [6, 5, 5]      # ties -> lower index
    assert make("bcc", (2, 2, 2), [0.3, 0.3, 0.4], 1).n_per_species == [5, 5, 6]            # 4.8 4.8 6.4 -> rem .8 .8 .4
    with pytest.raises(ValueError):
        make("bcc", (1, 1, 1), [0.9, 0.05, 0.05], 1)                                          # a species with 0 atoms
    with pytest.raises(ValueError):
        make("bcc", (2, 2, 2), [0.5, 0.4], 1)                                                 # does not sum to 1


# ------------------------------------------------------------------ D4-D5: counts, alpha; closed forms
def ordered(lattice, dims, rule):
    A = 4 if lattice == "fcc" else 2
    n = A * int(np.prod(dims))
    return np.array([rule(site % A) for site in range(n)], dtype=np.uint8)


def test_closed_form_B2():
    o = make("bcc", (4, 4, 4), [0.5, 0.5], 3)
    al = o.alpha(o.pair_counts(ordered("bcc", (4, 4, 4), lambda b: b)))
    np.testing.assert_array_equal(al[0], [[1, -1], [-1, 1]])
    for s in (1, 2):
        np.testing.assert_array_equal(al[s], [[-1, 1], [1, -1]])


def test_closed_form_L12():
    o = make("fcc", (4, 4, 4), [0.25, 0.75], 3)
    al = o.alpha(o.pair_counts(ordered("fcc", (4, 4, 4), lambda b: 0 if b == 0 else 1)))
    for s in (0, 2):
        np.testing.assert_allclose(al[s], [[1, -1 / 3], [-1 / 3, 1 / 9]], rtol=0, atol=1e-15)
    np.testing.assert_allclose(al[1], [[-3, 1], [1, -1 / 3]], rtol=0, atol=1e-15)


def test_closed_form_L10():
    o = make("fcc", (4, 4, 4), [0.5, 0.5], 3)
    al = o.alpha(o.pair_counts(ordered("fcc", (4, 4, 4), lambda b: 0 if b < 2 else 1)))
    for s in (0, 2):
        np.testing.assert_allclose(al[s], [[1 / 3, -1 / 3], [-1 / 3, 1 / 3]], rtol=0, atol=1e-15)
    np.testing.assert_array_equal(al[1], [[-1, 1], [1, -1]])


def test_objective_closed_forms():
    # B2 configuration against the B2 target -> J = 0; against target 0 -> sum_s w_s * 4 * 1
    tB2 = np.array([[[1, -1], [-1, 1]], [[-1, 1], [1, -1]], [[-1, 1], [1, -1]]], dtype=float)
    occ = ordered("bcc", (4, 4, 4), lambda b: b)
    o = make("bcc", (4, 4, 4), [0.5, 0.5], 3, w=[1.0, 0.5, 0.25], target=tB2)
    assert o.objective(o.pair_counts(occ)) == 0.0
    o0 = make("bcc", (4, 4, 4), [0.5, 0.5], 3, w=[1.0, 0.5, 0.25])
    assert o0.objective(o0.pair_counts(occ)) == 4.0 * (1.0 + 0.5 + 0.25)
    # a non-symmetric target distinguishes t_ij from t_ji: alpha(B2, shell 1) = [[1,-1],[-1,1]]
    t = np.zeros((1, 2, 2)); t[0, 0, 1] = 0.5
    o1 = make("bcc", (4, 4, 4), [0.5, 0.5], 1, w=[2.0], target=t)
    assert o1.objective(o1.pair_counts(occ)) == 2.0 * (1 + 2.25 + 1 + 1)


def test_single_species_alpha_zero():
    o = make("fcc", (3, 3, 3), [1.0], 3)
    c = o.pair_counts(np.zeros(o.N, dtype=np.uint8))
    assert (o.alpha(c) == 0).all() and o.objective(c) == 0.0
    assert c.reshape(-1).tolist() == [12 * o.N, 6 * o.N, 24 * o.N]


@pytest.mark.parametrize("lattice,dims,conc,S", [("fcc", (5, 5, 5), [0.2] * 5, 3), ("bcc", (6, 5, 4), [0.25] * 4, 3),
                                                 ("fcc", (3, 4, 5), [0.4, 0.4, 0.1, 0.1], 2),
                                                 ("bcc", (2, 2, 2), [0.5, 0.25, 0.25], 3)])
def test_sum_rules(lattice, dims, conc, S):
    o = make(lattice, dims, conc, S)
    occ = o.init_random(3, seed=99)
    for c in range(3):
        assert np.bincount(occ[c], minlength=o.M).tolist() == o.n_per_species          # composition exact
        n = o.pair_counts(occ[c]).astype(np.int64)
        al = o.alpha(n)
        cj = np.array(o.n_per_species) / o.N
        for s in range(S):
            assert (n[s].sum(1) == o.z[s] * np.array(o.n_per_species)).all()            # sum_j N_ij = z N_i
            assert (n[s] == n[s].T).all()                                               # N_ij = N_ji
            assert n[s].sum() == o.z[s] * o.N
            np.testing.assert_allclose(al[s] @ cj, 0, atol=1e-13)                       # sum_j c_j alpha_ij = 0
            np.testing.assert_array_equal(al[s], al[s].T)                               # alpha symmetric (A17)
            # the definition, retyped: alpha = 1 - (N_ij / (z N_i)) / c_j
            P = n[s] / (o.z[s] * np.array(o.n_per_species)[:, None])
            np.testing.assert_allclose(al[s], 1 - P / cj[None, :], rtol=0, atol=1e-13)


def test_pair_counts_equal_python_double_loop():
    o = make("fcc", (3, 3, 2), [0.5, 0.25, 0.25], 3)
    occ = o.init_random(1, seed=5)[0]
    want = np.zeros((3, 3, 3), dtype=np.int64)
    for s in range(3):
        tab = o.neighbor_table(s)
        for a in range(o.N):
            for v in tab[a]:
                want[s, occ[a], occ[v]] += 1
    np.testing.assert_array_equal(o.pair_counts(occ), want)


@pytest.mark.parametrize("lattice,dims,conc,S", [("fcc", (5, 4, 3), [0.2] * 5, 3), ("bcc", (4, 5, 6), [0.25] * 4, 3),
                                                 ("fcc", (1, 1, 1), [0.5, 0.5], 3), ("bcc", (1, 2, 3), [0.5, 0.5], 3),
                                                 ("fcc", (2, 2, 2), [0.125] * 8, 3), ("bcc", (2, 2, 2), [0.5, 0.25, 0.25], 3)])
def test_half_shell_identity_of_the_sorted_offset_list(lattice, dims, conc, S):
    """The fact the table-free recount kernel rests on, pinned on the oracle's table with numpy only:
    in the D2 order entry z-1-k of a shell is the reverse of entry k (following k and then z-1-k returns to the start
    site, on every cell size), hence the counts H over the second half of each shell give N = H + H^T, multi-edges and
    self-neighbours of tiny cells included."""
    o = make(lattice, dims, conc, S)
    occ = o.init_random(2, seed=21)
    for s in range(S):
        tab = o.neighbor_table(s).astype(np.int64)
        z = o.z[s]
        for k in range(z):
            np.testing.assert_array_equal(tab[tab[:, k], z - 1 - k], np.arange(o.N))
        for c in range(2):
            H = np.zeros((o.M, o.M), dtype=np.int64)
            for k in range(z // 2, z):
                np.add.at(H, (occ[c], occ[c][tab[:, k]]), 1)
            np.testing.assert_array_equal(H + H.T, o.pair_counts(occ[c])[s])


# ------------------------------------------------------------------ D8: random start
def test_init_is_fisher_yates_with_pinned_philox():
    o = make("bcc", (3, 3, 3), [0.5, 0.5], 1)
    seed, chain0 = 0x1234567887654321, 5
    occ = o.init_random(2, seed=seed, chain0=chain0)
    for c in range(2):
        ref = [0] * 27 + [1] * 27
        for n in range(o.N - 1, 0, -1):
            r = int(ho.philox4x32_10([n, 0, 0xFFFFFFFF, chain0 + c], [seed & 0xFFFFFFFF, seed >> 32])[0])
            j = (r * (n + 1)) >> 32
            ref[n], ref[j] = ref[j], ref[n]
        assert occ[c].tolist() == ref


def test_random_start_expectation_A18():
    # exact-composition shuffle, distinct neighbours: E[alpha_ij] = -1/(N-1) (i != j), E[alpha_ii] = (N-N_i)/(N_i (N-1))
    o = make("fcc", (3, 3, 3), [0.5, 0.25, 0.25], 2)
    n_chains = 3000
    occ = o.init_random(n_chains, seed=2024)
    counts, alpha, _ = o.sro_full(occ, n_threads=4)
    mean = alpha.mean(0)
    sem = alpha.std(0) / math.sqrt(n_chains)
    N, Ni = o.N, np.array(o.n_per_species)
    want = np.full((o.M, o.M), -1.0 / (N - 1))
    want[np.diag_indices(o.M)] = (N - Ni) / (Ni * (N - 1))
    for s in range(2):
        assert (np.abs(mean[s] - want) < 4.5 * sem[s] + 1e-12).all(), (mean[s], want, sem[s])
    # and the expectation is NOT zero at this size: the diagonal offset is resolved
    assert (np.abs(want[np.diag_indices(o.M)]) > 5 * sem[0][np.diag_indices(o.M)]).all()


# ------------------------------------------------------------------ D9.2: delta == recount difference
@pytest.mark.parametrize("lattice,dims,conc,S", [("bcc", (2, 2, 2), [0.5, 0.5], 3), ("fcc", (1, 1, 1), [0.5, 0.5], 3),
                                                 ("fcc", (2, 2, 2), [0.25] * 4, 3), ("bcc", (1, 2, 3), [0.5, 0.25, 0.25], 3),
                                                 ("fcc", (3, 3, 3), [0.2] * 5 if False else [0.25] * 4, 3),
                                                 ("bcc", (3, 3, 3), [0.5, 0.5], 3), ("fcc", (2, 1, 3), [0.5, 0.5], 2)])
def test_delta_equals_recount_for_all_unlike_pairs(lattice, dims, conc, S):
    o = make(lattice, dims, conc, S)
    occ = o.init_random(1, seed=3)[0]
    base = o.pair_counts(occ)
    pairs = [(a, b) for a in range(o.N) for b in range(o.N) if a != b and occ[a] != occ[b]]
    if len(pairs) > 3000:
        rng = np.random.default_rng(0)
        pairs = [pairs[i] for i in rng.choice(len(pairs), 3000, replace=False)]
    for a, b in pairs:
        swapped = occ.copy()
        swapped[a], swapped[b] = occ[b], occ[a]
        np.testing.assert_array_equal(o.delta_counts(occ, a, b, base), o.pair_counts(swapped))


# ------------------------------------------------------------------ brute force on a tiny cell
def test_brute_force_spectrum_bcc_2x2x2():
    # bcc 2x2x2 (N=16), shell 1, 8 A + 8 B, w = 1.  alpha_AB = 1 - N_AB/32, J = 4 alpha_AB^2 for target 0.
    o0 = make("bcc", (2, 2, 2), [0.5, 0.5], 1, w=[1.0])
    tB2 = np.array([[[1.0, -1.0], [-1.0, 1.0]]])
    oB = make("bcc", (2, 2, 2), [0.5, 0.5], 1, w=[1.0], target=tB2)
    spectrum, zeros_B2 = {}, 0
    for ones in itertools.combinations(range(16), 8):
        occ = np.zeros(16, dtype=np.uint8)
        occ[list(ones)] = 1
        c = o0.pair_counts(occ)
        J = o0.objective(c)
        spectrum[J] = spectrum.get(J, 0) + 1
        assert J == 4.0 * (1.0 - c[0, 0, 1] / 32.0) ** 2
        zeros_B2 += oB.objective(c) == 0.0
    assert zeros_B2 == 2
    assert spectrum == {0.0: 4900, 1 / 64: 6272, 1 / 4: 1568, 81 / 64: 128, 4.0: 2}


# ------------------------------------------------------------------ D9: MC dynamics
def py_propose(o, occ, seed, chain, step, k):
    """D9.1 restated with the pinned Philox."""
    r = [int(x) for x in ho.philox4x32_10([step & 0xFFFFFFFF, step >> 32, k, chain], [seed & 0xFFFFFFFF, seed >> 32])]
    N = o.N
    for r0, r1 in ((r[0], r[1]), (r[2], r[3])):
        a = (r0 * N) >> 32
        b = (r1 * (N - 1)) >> 32
        if b >= a:
            b += 1
        if occ[a] != occ[b]:
            return True, a, b
    return False, a, b


@pytest.mark.parametrize("lattice,dims,conc,S,K", [("bcc", (2, 2, 3), [0.5, 0.5], 2, 4), ("fcc", (2, 2, 2), [0.25] * 4, 3, 8),
                                                   ("bcc", (3, 3, 3), [0.5, 0.25, 0.25], 2, 5)])
def test_mc_step_is_lowest_index_improving_by_full_recount(lattice, dims, conc, S, K):
    """Exhaustive re-derivation of every step: proposals from the pinned Philox, every candidate's J from a
    FULL recount of the swapped configuration, lowest improving index applied."""
    M = len(conc)
    rng = np.random.default_rng(1)
    tgt = rng.uniform(-0.2, 0.2, size=(S, M, M))
    o = make(lattice, dims, conc, S, target=tgt)
    seed, chain0, step0, n_steps = 77, 3, (1 << 32) - 5, 40          # crosses the 32-bit step boundary
    occ = o.init_random(2, seed=seed, chain0=chain0)
    counts = np.stack([o.pair_counts(occ[c]) for c in range(2)])
    ref_occ = occ.copy()
    stats, log = o.mc_run(occ, counts, n_steps, K, seed, chain0=chain0, step0=step0, log_cap=64)
    total_acc = 0
    for c in range(2):
        x = ref_occ[c].copy()
        J_cur = o.objective(o.pair_counts(x))
        n_acc = n_null = 0
        h, moves, last = ho.HASH0, [], ho.NO_STEP
        for t in range(n_steps):
            step = step0 + t
            best = None
            for k in range(K):
                ok, a, b = py_propose(o, x, seed, chain0 + c, step, k)
                assert (ok, a, b) == o.propose(x, seed, chain0 + c, step, k)
                if not ok:
                    n_null += 1
                    continue
                y = x.copy()
                y[a], y[b] = x[b], x[a]
                Jk = o.objective(o.pair_counts(y))
                if best is None and Jk < J_cur:
                    best = (k, a, b, Jk)
            if best is not None:
                k, a, b, Jk = best
                x[a], x[b] = x[b], x[a]
                assert Jk < J_cur
                J_cur = Jk
                n_acc += 1
                last = step
                for word in (step & 0xFFFFFFFF, step >> 32, k, a, b):
                    h = ((h ^ word) * 0x100000001B3) & 0xFFFFFFFFFFFFFFFF
                moves.append((step, k, a, b))
        total_acc += n_acc
        np.testing.assert_array_equal(occ[c], x)
        np.testing.assert_array_equal(counts[c], o.pair_counts(x))          # incremental == recount at the end
        st = stats[c]
        assert (int(st["n_accept"]), int(st["n_null"]), int(st["hash"]), int(st["last_accept_step"])) == (n_acc, n_null, h, last)
        assert float(st["J"]) == J_cur
        got = [(int(m["step"]), int(m["k"]), int(m["a"]), int(m["b"])) for m in log[c][:n_acc]]
        assert got == moves[:64]
    assert total_acc > 0


def test_mc_invariances_split_run_chain_offset_eval_mode():
    w = wl.config(1)
    o = ho.Oracle(*w.create_args())
    occ0 = o.init_random(6, seed=w.seed)
    cnt0, _, _ = o.sro_full(occ0)
    # reference: all 6 chains, 400 steps in one go
    occ, cnt = occ0.copy(), cnt0.copy()
    st, _ = o.mc_run(occ, cnt, 400, w.K, w.seed, n_threads=3)
    # split run: 150 + 250 with step0, carrying stats
    occ_s, cnt_s = occ0.copy(), cnt0.copy()
    st_s, _ = o.mc_run(occ_s, cnt_s, 150, w.K, w.seed)
    st_s, _ = o.mc_run(occ_s, cnt_s, 250, w.K, w.seed, step0=150, stats=st_s)
    np.testing.assert_array_equal(occ, occ_s)
    np.testing.assert_array_equal(cnt, cnt_s)
    assert st.tobytes() == st_s.tobytes()
    # chains 2..5 alone via chain0, early-exit evaluation mode -> identical trajectories
    occ_c, cnt_c = occ0[2:].copy(), cnt0[2:].copy()
    st_c, _ = o.mc_run(occ_c, cnt_c, 400, w.K, w.seed, chain0=2, eval_all=False)
    np.testing.assert_array_equal(occ[2:], occ_c)
    assert st[2:].tobytes() == st_c.tobytes()
    # composition conserved, counts == recount, null fraction ~ (sum c_i^2)^2 = 0.04
    for c in range(6):
        assert np.bincount(occ[c], minlength=5).tolist() == [100] * 5
        np.testing.assert_array_equal(cnt[c], o.pair_counts(occ[c]))
    frac = st["n_null"].sum() / (6 * 400 * w.K)
    assert 0.03 < frac < 0.05


def test_mc_objective_monotone():
    w = wl.config(2, n_chains=1)
    o = ho.Oracle(*w.create_args())
    occ = o.init_random(1, seed=w.seed)
    cnt, _, J = o.sro_full(occ)
    prev, st = J[0], None
    for chunk in range(20):
        n_before = 0 if st is None else int(st["n_accept"][0])
        st, _ = o.mc_run(occ, cnt, 10, w.K, w.seed, step0=10 * chunk, stats=st)
        Jn = float(st["J"][0])
        if int(st["n_accept"][0]) > n_before:
            assert Jn < prev
        else:
            assert Jn == prev
        assert Jn == o.objective(o.pair_counts(occ[0]))
        prev = Jn


# ------------------------------------------------------------------ advisory cross-check (independent implementation)
def _golden_records():
    recs, targets = [], {}
    for line in open(os.path.join(GOLDEN, "survey_crosscheck.txt")):
        if not line.strip() or line[0] == "#":
            continue
        f = line.split()
        if f[0] in ("t3", "t4"):
            targets[f[0]] = [float(x) for x in f[1:]]
        else:
            recs.append(f)
    return recs, targets


def test_survey_crosscheck_targets():
    _, targets = _golden_records()
    assert wl.config(3).target[0, 0].tolist() == targets["t3"]
    assert wl.config(4).target[0, 0].tolist() == targets["t4"]
    for i in (3, 4):
        w = wl.config(i)
        np.testing.assert_allclose(w.target[0] @ np.array(w.conc), 0, atol=1e-16)
        assert (w.target[1:] == 0).all() and (w.target[0] == w.target[0].T).all()


@pytest.mark.parametrize("rec", _golden_records()[0], ids=lambda r: "-".join(r[:3]))
def test_survey_crosscheck_trajectories(rec):
    name, chain, n_steps = rec[0], int(rec[1]), int(rec[2])
    w = wl.config(int(name[1]))
    o = ho.Oracle(*w.create_args())
    occ = o.init_random(1, seed=w.seed, chain0=chain)
    cnt, _, J = o.sro_full(occ)
    if rec[3] != "-":
        assert J[0] == float(rec[3])
    st, log = o.mc_run(occ, cnt, n_steps, w.K, w.seed, chain0=chain, log_cap=8, eval_all=False)
    assert int(st["n_accept"][0]) == int(rec[4])
    assert int(st["n_null"][0]) == int(rec[5])
    assert float(st["J"][0]) == float(rec[6])
    assert int(st["hash"][0]) == int(rec[7], 16)
    for i, mv in enumerate(rec[8:]):
        s, k, a, b = (int(x) for x in mv.split(":"))
        m = log[0][i]
        assert (int(m["step"]), int(m["k"]), int(m["a"]), int(m["b"])) == (s, k, a, b)


# ---- best-of-K selection (Eq. 6) and search-depth termination (Alg. 3)
@pytest.mark.parametrize("lattice,dims,conc,S,K", [("bcc", (2, 2, 3), [0.5, 0.5], 2, 6), ("fcc", (2, 2, 2), [0.25] * 4, 3, 8),
                                                   ("bcc", (3, 3, 3), [0.5, 0.25, 0.25], 2, 5)])
@pytest.mark.parametrize("depth_limit", [0, 3])
def test_mc_ex_best_of_K_and_depth_by_full_recount(lattice, dims, conc, S, K, depth_limit):
    """Every step re-derived in Python: proposals from the pinned Philox, every candidate's J from a FULL recount, the
    minimum J (ties -> lowest k) applied iff it improves; depth = consecutive steps without a move; stop at the limit."""
    M = len(conc)
    rng = np.random.default_rng(2)
    tgt = rng.uniform(-0.2, 0.2, size=(S, M, M))
    o = make(lattice, dims, conc, S, target=tgt)
    seed, chain0, step0, n_steps = 91, 5, 17, 60
    occ = o.init_random(2, seed=seed, chain0=chain0)
    counts = np.stack([o.pair_counts(occ[c]) for c in range(2)])
    ref_occ = occ.copy()
    stats, log, depth, steps_done = o.mc_run_ex(occ, counts, n_steps, K, seed, chain0=chain0, step0=step0, log_cap=64,
                                                select_best=True, depth_limit=depth_limit)
    for c in range(2):
        x = ref_occ[c].copy()
        J_cur = o.objective(o.pair_counts(x))
        n_acc = n_null = d = t_done = 0
        h, moves = ho.HASH0, []
        for t in range(n_steps):
            if depth_limit and d >= depth_limit:
                break
            step = step0 + t
            best = None
            for k in range(K):
                ok, a, b = py_propose(o, x, seed, chain0 + c, step, k)
                if not ok:
                    n_null += 1
                    continue
                y = x.copy()
                y[a], y[b] = x[b], x[a]
                Jk = o.objective(o.pair_counts(y))
                if Jk < J_cur and (best is None or Jk < best[3]):
                    best = (k, a, b, Jk)
            if best is not None:
                k, a, b, Jk = best
                x[a], x[b] = x[b], x[a]
                J_cur = Jk
                n_acc += 1
                d = 0
                for word in (step & 0xFFFFFFFF, step >> 32, k, a, b):
                    h = ((h ^ word) * 0x100000001B3) & 0xFFFFFFFFFFFFFFFF
                moves.append((step, k, a, b))
            else:
                d += 1
            t_done = t + 1
        np.testing.assert_array_equal(occ[c], x)
        np.testing.assert_array_equal(counts[c], o.pair_counts(x))
        st = stats[c]
        assert (int(st["n_accept"]), int(st["n_null"]), int(st["hash"])) == (n_acc, n_null, h)
        assert float(st["J"]) == J_cur
        assert (int(depth[c]), int(steps_done[c])) == (d, t_done)
        got = [(int(m["step"]), int(m["k"]), int(m["a"]), int(m["b"])) for m in log[c][:n_acc]]
        assert got == moves[:64]
        if depth_limit:
            assert t_done < n_steps and d == depth_limit          # these small cells do stall within 60 steps


def test_mc_ex_reduces_to_the_north_star_rule_and_continues_exactly():
    o = make("fcc", (3, 3, 3), [0.5, 0.25, 0.25], 2, target=None)
    seed, K = 5, 12
    occ0 = o.init_random(3, seed=seed)
    cnt0 = np.stack([o.pair_counts(occ0[c]) for c in range(3)])
    # select_best = False, no depth limit == ora_mc_run
    a_occ, a_cnt = occ0.copy(), cnt0.copy()
    st_a, _ = o.mc_run(a_occ, a_cnt, 200, K, seed, eval_all=False)
    b_occ, b_cnt = occ0.copy(), cnt0.copy()
    st_b, _, _, done = o.mc_run_ex(b_occ, b_cnt, 200, K, seed)
    np.testing.assert_array_equal(a_occ, b_occ)
    assert (st_a["hash"] == st_b["hash"]).all() and (done == 200).all()
    # a split run with the depth carried over equals one run (best-of-K, depth limit 25)
    c_occ, c_cnt = occ0.copy(), cnt0.copy()
    st_c, _, d_c, done_c = o.mc_run_ex(c_occ, c_cnt, 400, K, seed, select_best=True, depth_limit=25)
    d_occ, d_cnt = occ0.copy(), cnt0.copy()
    st_d, _, d_d, done_1 = o.mc_run_ex(d_occ, d_cnt, 150, K, seed, select_best=True, depth_limit=25)
    st_d, _, d_d, done_2 = o.mc_run_ex(d_occ, d_cnt, 250, K, seed, step0=150, stats=st_d, select_best=True, depth_limit=25, depth=d_d)
    np.testing.assert_array_equal(c_occ, d_occ)
    assert (st_c["hash"] == st_d["hash"]).all() and (st_c["J"] == st_d["J"]).all()
    # a chain that stopped in the first part does nothing in the second; the others add up
    assert ((done_1 + done_2 == done_c) | (done_1 < 150)).all() and (d_c == d_d).all()
    # best-of-K never does worse in one step than lowest-index from the same state
    e_occ, e_cnt = occ0.copy(), cnt0.copy()
    st_e, _, _, _ = o.mc_run_ex(e_occ, e_cnt, 1, K, seed, select_best=True)
    f_occ, f_cnt = occ0.copy(), cnt0.copy()
    st_f, _ = o.mc_run(f_occ, f_cnt, 1, K, seed, eval_all=False)
    assert (st_e["J"] <= st_f["J"]).all()


# ---- the selection step of the global search (Alg. 1)
def test_pool_select_keeps_the_best_and_reseeds_the_rest():
    o = make("bcc", (3, 3, 3), [0.5, 0.25, 0.25], 2, target=None)
    seed, C, K, n_keep = 8, 12, 8, 5
    occ = o.init_random(C, seed=seed)
    counts = np.stack([o.pair_counts(occ[c]) for c in range(C)])
    stats, _ = o.mc_run(occ, counts, 30, K, seed, eval_all=False)
    occ[7], counts[7], stats[7] = occ[2], counts[2], stats[2]              # an exact tie between slots 2 and 7
    J = np.array([o.objective(counts[c]) for c in range(C)])
    occ0, cnt0, st0 = occ.copy(), counts.copy(), stats.copy()
    order = o.pool_select(occ, counts, stats, n_keep, seed=99, new_chain0=1000)
    # kept = the n_keep smallest J, ascending, ties by index; nothing kept is worse than anything dropped
    assert len(set(order.tolist())) == n_keep
    kept_J = J[order]
    assert (np.diff(kept_J) >= 0).all()
    dropped = [c for c in range(C) if c not in set(order.tolist())]
    assert kept_J.max() <= J[dropped].min()
    for r in range(n_keep - 1):
        if kept_J[r] == kept_J[r + 1]:
            assert order[r] < order[r + 1]
    if 2 in order.tolist() and 7 in order.tolist():
        assert order.tolist().index(2) + 1 == order.tolist().index(7)
    for r, c in enumerate(order):
        np.testing.assert_array_equal(occ[r], occ0[c])
        np.testing.assert_array_equal(counts[r], cnt0[c])
        assert stats[r] == st0[c]
    # the rest: fresh D8 configurations with the new chain ids, recounted, stats reset
    np.testing.assert_array_equal(occ[n_keep:], o.init_random(C - n_keep, 99, 1000))
    for c in range(n_keep, C):
        np.testing.assert_array_equal(counts[c], o.pair_counts(occ[c]))
    assert (stats[n_keep:] == ho.fresh_stats(C - n_keep)).all()
