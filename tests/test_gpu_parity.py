"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same seeded
inputs.  Bar (BASELINE.json:north_star): pair counts, occupancies, accepted-move sequences, n_accept, n_null
bit-exact; J within 1e-12 relative (it is expected, and asserted, to be bit-equal under D6)."""
import numpy as np
import pytest

from oracle import hea_oracle as ho
from paper_2411_18906_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def pair(hb, w):
    return hb.Hea(*w.create_args()), ho.Oracle(*w.create_args())


def small(lattice, dims, conc, S, target_seed=None, rng=(-0.1, 0.1), **kw):
    base = dict(name="t", lattice=lattice, dims=dims, conc=conc, n_shells=S, shell_w=[1.0, 0.5, 0.25][:S],
                n_chains=4, n_steps=50, K=8, seed=42, target_seed=target_seed, target_range=rng)
    base.update(kw)
    return wl.Workload(**base)


def assert_stats_equal(got, want):
    for f in ("n_accept", "n_null", "hash", "last_accept_step"):
        np.testing.assert_array_equal(got[f], want[f], err_msg=f)
    np.testing.assert_allclose(got["J"], want["J"], rtol=1e-12, atol=0)
    np.testing.assert_array_equal(got["J"], want["J"])            # bit-equal under the fixed D6 order


LATTICES = [("fcc", (3, 3, 3), [0.5, 0.5], 3), ("fcc", (3, 4, 5), [0.2] * 5, 3), ("bcc", (4, 3, 5), [0.25] * 4, 3),
            ("bcc", (3, 3, 3), [0.5, 0.25, 0.25], 2), ("fcc", (1, 1, 1), [0.5, 0.5], 3), ("bcc", (1, 2, 3), [0.5, 0.5], 3),
            ("fcc", (2, 2, 2), [0.125] * 8, 3), ("bcc", (7, 7, 7), [1 / 7] * 7, 1), ("fcc", (6, 5, 4), [0.4, 0.4, 0.1, 0.1], 2),
            ("bcc", (2, 2, 2), [1.0], 3), ("fcc", (4, 4, 4), [1 / 6] * 6, 3), ("bcc", (5, 5, 5), [0.2, 0.3, 0.5], 3)]


@pytest.mark.parametrize("lattice,dims,conc,S", LATTICES)
def test_info_and_neighbor_table(hb, lattice, dims, conc, S):
    h, o = pair(hb, small(lattice, dims, conc, S))
    assert (h.N, h.z, h.n_per_species) == (o.N, o.z, o.n_per_species)
    for s in range(S):
        np.testing.assert_array_equal(h.neighbor_table(s), o.neighbor_table(s))


SRO_ENGINES = [1, 2]          # 1 = table-driven (hea_sro.cu), 2 = table-free stencil (hea_sro2.cu); 0 = auto picks 2


@pytest.mark.parametrize("engine", SRO_ENGINES)
@pytest.mark.parametrize("lattice,dims,conc,S", LATTICES)
def test_init_and_sro_full_bit_exact(hb, lattice, dims, conc, S, engine):
    w = small(lattice, dims, conc, S, target_seed=3)
    h, o = pair(hb, w)
    h.set_option("sro_engine", engine)
    B = 5
    occ = h.init_random(B, seed=w.seed, chain0=7)
    want_occ = o.init_random(B, seed=w.seed, chain0=7)
    np.testing.assert_array_equal(occ.cpu().numpy(), want_occ)
    counts, alpha, obj = h.sro_full(occ)
    wc, wa, wj = o.sro_full(want_occ)
    np.testing.assert_array_equal(counts.cpu().numpy(), wc)
    np.testing.assert_array_equal(alpha.cpu().numpy(), wa)
    np.testing.assert_array_equal(obj.cpu().numpy(), wj)


@pytest.mark.parametrize("lattice,dims,conc", [("fcc", (40, 40, 40), [0.25] * 4), ("bcc", (30, 20, 25), [0.2] * 5),
                                               ("fcc", (37, 41, 43), [0.4, 0.4, 0.1, 0.1]), ("bcc", (3, 2, 2), [0.5, 0.5])])
def test_init_random_large_cells_bit_exact(hb, lattice, dims, conc):
    # D8 at sizes where the kernel applies groups of 32 commuting swaps in parallel (shared-memory and global-memory
    # configurations): the occupancies must equal the oracle's serial Fisher-Yates byte for byte
    w = small(lattice, dims, conc, 2)
    h, o = pair(hb, w)
    occ = h.init_random(3, seed=77, chain0=5)
    np.testing.assert_array_equal(occ.cpu().numpy(), o.init_random(3, seed=77, chain0=5))


@pytest.mark.parametrize("engine", SRO_ENGINES)
def test_sro_full_ordered_structures(hb, engine):
    # B2 on bcc: closed form alpha (+1/-1), through the GPU path
    w = small("bcc", (6, 6, 6), [0.5, 0.5], 3)
    h, o = pair(hb, w)
    h.set_option("sro_engine", engine)
    import torch
    occ = torch.tensor(np.arange(h.N, dtype=np.int64) % 2, dtype=torch.uint8, device="cuda").reshape(1, -1)
    counts, alpha, obj = h.sro_full(occ)
    al = alpha.cpu().numpy()[0]
    np.testing.assert_array_equal(al[0], [[1, -1], [-1, 1]])
    np.testing.assert_array_equal(al[1], [[-1, 1], [1, -1]])
    np.testing.assert_array_equal(counts.cpu().numpy()[0], o.pair_counts(occ.cpu().numpy()[0]))


@pytest.mark.parametrize("engine", SRO_ENGINES)
@pytest.mark.parametrize("L,B", [(10, 3), (16, 2), (23, 1)])
def test_sro_full_multi_tile_and_ragged(hb, L, B, engine):
    # several blocks / grid-stride iterations, flushes of the 16-bit accumulators, N % 4 != 0 for bcc odd L
    for lattice, conc in (("fcc", [0.2] * 5), ("bcc", None)):
        if conc is None:
            n = 2 * L ** 3
            conc = [0.5, 0.25, 0.25] if n % 4 == 0 else [0.5, 0.5]
        w = small(lattice, (L, L, L), conc, 3, target_seed=9)
        h, o = pair(hb, w)
        h.set_option("sro_engine", engine)
        occ = h.init_random(B, seed=5)
        counts, alpha, obj = h.sro_full(occ)
        wc, wa, wj = o.sro_full(occ.cpu().numpy(), n_threads=4)
        np.testing.assert_array_equal(counts.cpu().numpy(), wc)
        np.testing.assert_array_equal(obj.cpu().numpy(), wj)


@pytest.mark.parametrize("lattice,dims,conc,S", [("fcc", (17, 9, 45), [0.2] * 5, 3), ("bcc", (9, 21, 35), [0.25] * 4, 3),
                                                 ("fcc", (8, 8, 33), [0.5, 0.25, 0.25], 2), ("bcc", (11, 3, 70), [1 / 7] * 7, 3),
                                                 ("fcc", (2, 13, 1), [0.5, 0.5], 3), ("fcc", (12, 10, 21), [0.125] * 8, 3)])
@pytest.mark.parametrize("tile_xy,tile_z,lanes,threads", [(0, 0, 0, 0), (1, 12, 1, 0), (3, 22, 2, 384), (8, 34, 1, 128),
                                                          (5, 12, 2, 256), (8, 34, 2, 0), (8, 22, 1, 0)])
def test_sro_stencil_tilings(hb, lattice, dims, conc, S, tile_xy, tile_z, lanes, threads):
    # the stencil engine over every row-pitch variant, ragged last tiles in all three directions, tiles smaller and
    # larger than the cell, z extents above one tile; the table engine and the oracle must both agree
    w = small(lattice, dims, conc, S, target_seed=4)
    h, o = pair(hb, w)
    occ = h.init_random(3, seed=11)
    h.set_option("sro_engine", 1)
    c_tab, _, _ = h.sro_full(occ)
    h.set_option("sro_engine", 2)
    h.set_option("sro_tile_xy", tile_xy)
    h.set_option("sro_tile_z", tile_z)
    h.set_option("sro_lanes", lanes)
    h.set_option("sro_threads", threads)
    c_st, _, j_st = h.sro_full(occ)
    wc, _, wj = o.sro_full(occ.cpu().numpy(), n_threads=4)
    np.testing.assert_array_equal(c_st.cpu().numpy(), wc)
    np.testing.assert_array_equal(c_tab.cpu().numpy(), wc)
    np.testing.assert_array_equal(j_st.cpu().numpy(), wj)


@pytest.mark.parametrize("bps,flush", [(1, 2), (1, 0), (4, 1), (0, 3)])
def test_sro_stencil_blocks_spanning_configurations_and_flushes(hb, bps, flush):
    # 40 configurations x 18 tiles over 148..592 persistent blocks: blocks cross configuration boundaries in the middle
    # of their item range and unpack their packed rows every `flush` tiles
    w = small("fcc", (20, 20, 40), [0.2] * 5, 3, target_seed=6)
    h, o = pair(hb, w)
    occ = h.init_random(40, seed=13)
    h.set_option("sro_engine", 2)
    h.set_option("sro_blocks_per_sm", bps)
    h.set_option("sro_flush_tiles", flush)
    counts, _, obj = h.sro_full(occ)
    wc, _, wj = o.sro_full(occ.cpu().numpy(), n_threads=8)
    np.testing.assert_array_equal(counts.cpu().numpy(), wc)
    np.testing.assert_array_equal(obj.cpu().numpy(), wj)


@pytest.mark.parametrize("conc", [[0.01, 0.01, 0.01, 0.01, 0.96], [0.96, 0.01, 0.01, 0.01, 0.01], [0.02, 0.02, 0.02, 0.94],
                                  [0.005] * 7 + [0.965], [1.0]])
@pytest.mark.parametrize("tile_z,lanes", [(12, 2), (22, 2), (34, 2), (22, 1)])
def test_sro_stencil_packed_field_capacity(hb, conc, tile_z, lanes):
    # nearly pure configurations drive single packed fields to their maximum (12 per site and shell): long item ranges
    # per block (one block per SM) must unpack before any field of the per-thread rows overflows
    w = small("fcc", (16, 16, 80), conc, 3, target_seed=6)
    h, o = pair(hb, w)
    occ = h.init_random(6, seed=17)
    h.set_option("sro_engine", 2)
    h.set_option("sro_blocks_per_sm", 1)
    h.set_option("sro_tile_z", tile_z)
    h.set_option("sro_lanes", lanes)
    counts, _, obj = h.sro_full(occ)
    wc, _, wj = o.sro_full(occ.cpu().numpy(), n_threads=8)
    np.testing.assert_array_equal(counts.cpu().numpy(), wc)
    np.testing.assert_array_equal(obj.cpu().numpy(), wj)


def test_sro_stencil_unaligned_occupancy_falls_back_to_table_kernel(hb):
    import torch
    w = small("fcc", (6, 6, 6), [0.2] * 5, 3, target_seed=6)
    h, o = pair(hb, w)
    occ = h.init_random(2, seed=3)
    buf = torch.zeros(occ.numel() + 8, dtype=torch.uint8, device="cuda")
    shifted = buf[1:1 + occ.numel()].view(2, -1)
    shifted.copy_(occ)
    assert shifted.data_ptr() % 4 == 1
    counts, _, _ = h.sro_full(shifted)                       # auto: table kernel (another CUDA kernel, no CPU path)
    np.testing.assert_array_equal(counts.cpu().numpy(), o.sro_full(occ.cpu().numpy())[0])
    h.set_option("sro_engine", 2)
    with pytest.raises(hb.HeaError):
        h.sro_full(shifted)


def test_sro_stencil_full_size_sweep_point(hb):
    # configs[4] at its largest cell in the launch configuration the sweep times (fcc 100^3, 5 species, 3 shells):
    # stencil == table engine on every count, and == the oracle
    w = small("fcc", (100, 100, 100), [0.2] * 5, 3, target_seed=2)
    h, o = pair(hb, w)
    occ = h.init_random(2, seed=5)
    h.set_option("sro_engine", 1)
    c_tab, _, _ = h.sro_full(occ)
    h.set_option("sro_engine", 2)
    c_st, _, j_st = h.sro_full(occ)
    np.testing.assert_array_equal(c_st.cpu().numpy(), c_tab.cpu().numpy())
    wc, _, wj = o.sro_full(occ.cpu().numpy(), n_threads=8)
    np.testing.assert_array_equal(c_st.cpu().numpy(), wc)
    np.testing.assert_array_equal(j_st.cpu().numpy(), wj)


def run_both(hb, w, n_chains, n_steps, log_cap=16, chain0=0, step0=0, opts=None, threads=8):
    h, o = pair(hb, w)
    for k, v in (opts or {}).items():
        h.set_option(k, v)
    occ = h.init_random(n_chains, seed=w.seed, chain0=chain0)
    counts, _, _ = h.sro_full(occ, want_alpha=False, want_obj=False)
    o_occ = occ.cpu().numpy().copy()
    o_cnt = counts.cpu().numpy().copy()
    stats, log = h.mc_run(occ, counts, n_steps, w.K, w.seed, chain0=chain0, step0=step0, log_cap=log_cap)
    o_stats, o_log = o.mc_run(o_occ, o_cnt, n_steps, w.K, w.seed, chain0=chain0, step0=step0, log_cap=log_cap,
                              n_threads=threads, eval_all=False)
    np.testing.assert_array_equal(occ.cpu().numpy(), o_occ)
    np.testing.assert_array_equal(counts.cpu().numpy(), o_cnt)
    assert_stats_equal(hb.stats_to_numpy(stats), o_stats)
    if log_cap:
        got = hb.log_to_numpy(log)
        for c in range(n_chains):
            n = min(int(o_stats["n_accept"][c]), log_cap)
            for f in ("step", "k", "a", "b"):
                np.testing.assert_array_equal(got[c][:n][f], o_log[c][:n][f])
    # the incremental counts equal a fresh recount of the final configuration
    recount, _, obj = h.sro_full(occ)
    np.testing.assert_array_equal(recount.cpu().numpy(), o_cnt)
    np.testing.assert_array_equal(obj.cpu().numpy(), o_stats["J"])
    return o_stats


@pytest.mark.parametrize("cluster", [1, 2, 5, 8])
@pytest.mark.parametrize("window", [0, 1, 3, 64])
@pytest.mark.parametrize("occ_mode", [1, 2, 3])
def test_mc_parity_all_launch_variants(hb, cluster, window, occ_mode):
    # results never depend on the launch shape: blocks per chain, speculative window cap, occupancy placement
    w = small("fcc", (4, 4, 4), [0.2, 0.2, 0.2, 0.4], 3, target_seed=5, K=24, n_steps=400)
    st = run_both(hb, w, 5, 400, opts={"mc_cluster": cluster, "mc_window": window, "mc_occ_mode": occ_mode})
    assert st["n_accept"].sum() > 50


@pytest.mark.parametrize("threads", [32, 64, 256, 1024])
@pytest.mark.parametrize("cluster", [1, 4])
@pytest.mark.parametrize("neighbors", [1, 2])
def test_mc_parity_block_sizes_reject_regime(hb, threads, cluster, neighbors):
    # target 0 on a small cell converges quickly: long windows without a move, then rare moves inside windows
    w = small("bcc", (6, 6, 6), [0.25] * 4, 3, K=32, n_steps=3000)
    st = run_both(hb, w, 3, 3000, log_cap=256,
                  opts={"mc_threads": threads, "mc_cluster": cluster, "mc_neighbors": neighbors})
    assert (st["n_accept"] > 20).all()


@pytest.mark.parametrize("lattice,dims", [("fcc", (7, 5, 6)), ("bcc", (5, 8, 6)), ("fcc", (3, 3, 9)), ("bcc", (2, 7, 7))])
@pytest.mark.parametrize("occ_mode", [1, 2])
def test_mc_parity_interior_fast_path(hb, lattice, dims, occ_mode):
    # interior sites take neighbours as site + offset; boundary sites (and cells with an L < 3) use the table
    w = small(lattice, dims, [0.3, 0.3, 0.4], 3, target_seed=21, K=48, n_steps=300)
    run_both(hb, w, 4, 300, opts={"mc_neighbors": 2, "mc_occ_mode": occ_mode})


@pytest.mark.parametrize("lattice,dims,conc,S", LATTICES[:9])
def test_mc_parity_lattices_including_degenerate_cells(hb, lattice, dims, conc, S):
    w = small(lattice, dims, conc, S, target_seed=11, K=16)
    run_both(hb, w, 3, 80)


@pytest.mark.parametrize("K,threads", [(1, 0), (7, 32), (33, 64), (200, 0), (1024, 0), (64, 96)])
def test_mc_parity_candidate_counts(hb, K, threads):
    w = small("bcc", (5, 5, 5), [0.2, 0.3, 0.5], 3, target_seed=2, K=K)
    run_both(hb, w, 3, 40, opts={"mc_threads": threads})


# ---- halo engine (hea_mc2.cu): padded one-hot configuration, coordinate-based adjacency
@pytest.mark.parametrize("lattice,dims,conc,S", LATTICES[:9])
@pytest.mark.parametrize("occ_mode", [1, 2])
def test_mc_halo_engine_lattices_including_degenerate_cells(hb, lattice, dims, conc, S, occ_mode):
    if occ_mode == 2 and len(conc) > 4:
        pytest.skip("a nibble holds a one-hot code of at most 4 species")
    w = small(lattice, dims, conc, S, target_seed=11, K=16)
    run_both(hb, w, 3, 80, opts={"mc_engine": 2, "mc_occ_mode": occ_mode})


@pytest.mark.parametrize("threads", [32, 256, 1024])
@pytest.mark.parametrize("window", [0, 1, 3])
@pytest.mark.parametrize("occ_mode", [1, 2])
def test_mc_halo_engine_launch_variants(hb, threads, window, occ_mode):
    w = small("fcc", (4, 4, 4), [0.2, 0.2, 0.2, 0.4], 3, target_seed=5, K=24, n_steps=400)
    st = run_both(hb, w, 5, 400, opts={"mc_engine": 2, "mc_threads": threads, "mc_window": window, "mc_occ_mode": occ_mode})
    assert st["n_accept"].sum() > 50


@pytest.mark.parametrize("lattice,dims", [("fcc", (7, 5, 6)), ("bcc", (5, 8, 6)), ("fcc", (3, 3, 9)), ("bcc", (3, 7, 4))])
def test_mc_halo_engine_reject_regime_and_neighbouring_pairs(hb, lattice, dims):
    # target 0 on small cells: converges, then long windows; small cells make (a, b) neighbours often (exclusion term)
    w = small(lattice, dims, [0.25] * 4, 3, K=32, n_steps=2000)
    st = run_both(hb, w, 3, 2000, log_cap=256, opts={"mc_engine": 2})
    assert (st["n_accept"] > 10).all()


@pytest.mark.parametrize("team", [2, 5, 9])
@pytest.mark.parametrize("on_off", [(1, 1), (64, 32), (512, 128), (0, 0)])
@pytest.mark.parametrize("occ_mode", [1, 2])
def test_mc_halo_engine_teams(hb, team, on_off, occ_mode):
    # R blocks per chain through global memory; (1, 1) = always TEAM, small thresholds = frequent SOLO <-> TEAM switches
    w = small("fcc", (4, 4, 4), [0.2, 0.2, 0.2, 0.4], 3, target_seed=5, K=24, n_steps=600)
    opts = {"mc_engine": 2, "mc_team": team, "mc_occ_mode": occ_mode, "mc_threads": 64}
    if on_off[0]:
        opts.update({"mc_team_on": on_off[0], "mc_team_off": on_off[1]})
    st = run_both(hb, w, 5, 600, opts=opts)
    assert st["n_accept"].sum() > 50


@pytest.mark.parametrize("team,threads", [(4, 256), (9, 1024), (32, 32)])
def test_mc_halo_engine_teams_reject_regime(hb, team, threads):
    w = small("bcc", (6, 6, 6), [0.25] * 4, 3, K=32, n_steps=3000)
    st = run_both(hb, w, 3, 3000, log_cap=256, opts={"mc_engine": 2, "mc_team": team, "mc_threads": threads})
    assert (st["n_accept"] > 20).all()


@pytest.mark.parametrize("lattice,dims,conc,S,K", [("fcc", (4, 4, 4), [0.2, 0.2, 0.2, 0.4], 3, 24), ("bcc", (5, 5, 5), [0.2] * 5, 3, 70),
                                                   ("fcc", (3, 3, 3), [0.5, 0.5], 1, 33), ("bcc", (4, 4, 4), [1 / 8] * 8, 2, 128),
                                                   ("fcc", (2, 2, 2), [0.25] * 4, 3, 40), ("fcc", (5, 4, 3), [1 / 6] * 6, 3, 17)])
@pytest.mark.parametrize("threads,team", [(512, 1), (1024, 1), (1024, 3)])
@pytest.mark.parametrize("accept", [2, 3])
def test_mc_halo_engine_accept_engine(hb, lattice, dims, conc, S, K, threads, team, accept):
    # single-step windows run 8 lanes per candidate (T >= 512), accept = 3: pipelined over epochs with records computed
    # ahead (small cells make most records stale: the recompute path); same trajectory as thread-per-candidate and the oracle
    w = small(lattice, dims, conc, S, target_seed=9, K=K, n_steps=400, rng=(-0.2, 0.2))
    st = run_both(hb, w, 3, 400, log_cap=400, opts={"mc_engine": 2, "mc_threads": threads, "mc_team": team, "mc_accept": accept})
    assert st["n_accept"].sum() > 5


def test_mc_halo_engine_c3_c4_prefix(hb):
    st = run_both(hb, wl.config(3), 4, 300, log_cap=300, opts={"mc_engine": 2})
    assert (st["n_accept"] > 250).all()
    st = run_both(hb, wl.config(4), 3, 300, log_cap=300, opts={"mc_engine": 2})
    assert (st["n_accept"] > 250).all()


def test_mc_c1_full(hb):
    w = wl.config(1)                                        # 64 chains x 10,000 steps x K=32, target 0
    st = run_both(hb, w, w.n_chains, w.n_steps, log_cap=64)
    assert int(st["n_accept"][0]) == 53 and float(st["J"][0]) == 0.0     # SURVEY cross-check values


def test_mc_c2_prefix(hb):
    w = wl.config(2)
    run_both(hb, w, 32, 3000)


def test_mc_c3_prefix(hb):
    w = wl.config(3)
    st = run_both(hb, w, 8, 400, log_cap=400)
    assert (st["n_accept"] > 300).all()                    # accept regime


def test_mc_c4_prefix(hb):
    w = wl.config(4)
    st = run_both(hb, w, 4, 300, log_cap=300)
    assert (st["n_accept"] > 250).all()


def test_mc_c4_bench_launch_configuration_through_convergence(hb):
    # exactly what bench.py launches (16 chains -> teams of 9 blocks, 512 threads, accept engine, then TEAM windows),
    # through the accept regime (~70,000 steps), the transition and into the reject regime
    w = wl.config(4)
    st = run_both(hb, w, w.n_chains, 300_000, log_cap=64, threads=16)
    assert (st["n_accept"] > 60_000).all() and (st["last_accept_step"] < 90_000).all()


def test_mc_c3_many_chains_through_convergence(hb):
    w = wl.config(3)
    st = run_both(hb, w, 64, 6000, log_cap=64, threads=16)
    assert (st["n_accept"] > 1000).all()


def test_fig3_workflow_non_equiatomic_target_from_small_cell(hb):
    # SURVEY 8f-3 / PAPER.md Fig. 3: a 500-atom Fe40Mn40Cr10Co10 cell is refined, its measured alpha becomes the target
    # of the 256,000-atom cell; every stage GPU == oracle (exercises c_j != 1/M in g_ij and in the sum rule)
    ws = wl.fig3_small_workload(2000)
    h, o = pair(hb, ws)
    st = run_both(hb, ws, 1, 2000, log_cap=0)
    occ = h.init_random(1, seed=ws.seed)
    cnt, _, _ = h.sro_full(occ, want_alpha=False, want_obj=False)
    h.mc_run(occ, cnt, 2000, ws.K, ws.seed)
    _, alpha, _ = h.sro_full(occ, want_alpha=True)
    o_occ = o.init_random(1, ws.seed)
    o_cnt, _, _ = o.sro_full(o_occ)
    o.mc_run(o_occ, o_cnt, 2000, ws.K, ws.seed, eval_all=False)
    _, o_alpha, _ = o.sro_full(o_occ)
    a = alpha.cpu().numpy()
    np.testing.assert_array_equal(a, o_alpha)
    conc = np.asarray(ws.conc)
    np.testing.assert_allclose((a[0] * conc[None, None, :]).sum(-1), 0.0, atol=1e-12)       # sum_j c_j alpha_ij = 0
    np.testing.assert_array_equal(a[0], np.swapaxes(a[0], -1, -2))                            # alpha symmetric (A17)
    wlg = wl.fig3_large_workload(a[0], n_chains=4)
    st = run_both(hb, wlg, 4, 3000, log_cap=64, threads=4)
    assert (st["n_accept"] > 2000).all()


def test_mc_c4_global_occupancy_path(hb):
    w = wl.config(4)
    run_both(hb, w, 2, 100, opts={"mc_occ_mode": 3, "mc_cluster": 8})


def test_mc_split_run_and_chain_offset(hb):
    w = small("fcc", (5, 5, 5), [0.2] * 5, 2, K=32, seed=1)
    h, o = pair(hb, w)
    occ0 = h.init_random(6, seed=w.seed)
    cnt0, _, _ = h.sro_full(occ0, want_alpha=False, want_obj=False)
    occ, cnt = occ0.clone(), cnt0.clone()
    st, _ = h.mc_run(occ, cnt, 400, w.K, w.seed)
    occ_s, cnt_s = occ0.clone(), cnt0.clone()
    st_s, _ = h.mc_run(occ_s, cnt_s, 150, w.K, w.seed)
    st_s, _ = h.mc_run(occ_s, cnt_s, 250, w.K, w.seed, step0=150, stats=st_s)
    assert (occ == occ_s).all() and (cnt == cnt_s).all() and (st == st_s).all()
    occ_c, cnt_c = occ0[2:].clone(), cnt0[2:].clone()
    h.set_option("mc_cluster", 4)
    h.set_option("mc_threads", 64)
    st_c, _ = h.mc_run(occ_c, cnt_c, 400, w.K, w.seed, chain0=2)
    assert (occ[2:] == occ_c).all() and (st[2:] == st_c).all()


def test_mc_large_step_offset(hb):
    w = small("bcc", (4, 4, 4), [0.25] * 4, 3, target_seed=8, K=16)
    run_both(hb, w, 2, 60, step0=(1 << 32) - 20, chain0=(1 << 32) - 2)


def test_empty_and_zero_step_calls(hb):
    import torch
    w = small("bcc", (3, 3, 3), [0.5, 0.5], 2)
    h, o = pair(hb, w)
    occ = h.init_random(2, seed=1)
    counts, _, obj = h.sro_full(occ)
    before = occ.clone()
    st, _ = h.mc_run(occ, counts, 0, 8, 1)                   # zero steps: state unchanged, J reported
    assert (occ == before).all()
    np.testing.assert_array_equal(hb.stats_to_numpy(st)["J"], obj.cpu().numpy())
    empty = torch.empty((0, h.N), dtype=torch.uint8, device="cuda")
    c0, _, _ = h.sro_full(empty)
    assert c0.shape[0] == 0


def test_argument_errors(hb):
    w = small("bcc", (3, 3, 3), [0.5, 0.5], 2)
    h, _ = pair(hb, w)
    occ = h.init_random(1, seed=1)
    counts, _, _ = h.sro_full(occ)
    with pytest.raises(hb.HeaError) as e:
        h.mc_run(occ, counts, 1, 0, 1)
    assert e.value.code == hb.HEA_EINVAL
    with pytest.raises(hb.HeaError):
        h.mc_run(occ, counts, 1, 2000, 1)
    with pytest.raises(hb.HeaError):
        h.set_option("mc_cluster", 9)
    with pytest.raises(hb.HeaError):
        h.set_option("nonsense", 1)
    with pytest.raises(hb.HeaError) as e:
        hb.Hea("fcc", (2, 2, 2), [0.5, 0.4], [1.0], np.zeros((1, 2, 2)))
    assert e.value.code == hb.HEA_EINVAL
    with pytest.raises(hb.HeaError) as e:
        hb.Hea("fcc", (2, 2, 2), [1 / 9] * 9, [1.0], np.zeros((1, 9, 9)))
    assert e.value.code == hb.HEA_EUNSUPPORTED


def test_host_buffer_entry_points(hb):
    w = small("fcc", (6, 6, 6), [0.25] * 4, 2, target_seed=4, K=32)
    h, o = pair(hb, w)
    occ = o.init_random(6, seed=w.seed)
    counts, alpha, obj = h.sro_full_host(occ, want_alpha=True)
    wc, wa, wj = o.sro_full(occ)
    np.testing.assert_array_equal(counts, wc)
    np.testing.assert_array_equal(alpha, wa)
    np.testing.assert_array_equal(obj, wj)
    g_occ = occ.copy()
    g_counts, g_stats = h.mc_run_host(g_occ, 200, w.K, w.seed)
    o_cnt = wc.copy()
    o_stats, _ = o.mc_run(occ, o_cnt, 200, w.K, w.seed, n_threads=4)
    np.testing.assert_array_equal(g_occ, occ)
    np.testing.assert_array_equal(g_counts, o_cnt)
    assert_stats_equal(g_stats, o_stats)


# ---- hea_mc_run_ex (best-of-K selection, search-depth termination) against ora_mc_run_ex
def run_both_ex(hb, w, n_chains, n_steps, select_best, depth_limit, opts=None, log_cap=64, split=None):
    h, o = pair(hb, w)
    for k, v in (opts or {}).items():
        h.set_option(k, v)
    occ = h.init_random(n_chains, seed=w.seed)
    counts, _, _ = h.sro_full(occ, want_alpha=False, want_obj=False)
    o_occ, o_cnt = occ.cpu().numpy().copy(), counts.cpu().numpy().copy()
    o_stats, o_log, o_depth, o_done = o.mc_run_ex(o_occ, o_cnt, n_steps, w.K, w.seed, log_cap=log_cap,
                                                  select_best=select_best, depth_limit=depth_limit)
    if split is None:
        stats, log, depth, done = h.mc_run_ex(occ, counts, n_steps, w.K, w.seed, log_cap=log_cap,
                                              select_best=select_best, depth_limit=depth_limit)
        done = done.cpu().numpy().astype(np.uint64)
    else:                                                       # two calls, depth and stats carried over
        stats, log, depth, d1 = h.mc_run_ex(occ, counts, split, w.K, w.seed, log_cap=log_cap,
                                            select_best=select_best, depth_limit=depth_limit)
        stats, _, depth, d2 = h.mc_run_ex(occ, counts, n_steps - split, w.K, w.seed, step0=split, stats=stats,
                                          select_best=select_best, depth_limit=depth_limit, depth=depth)
        d1, d2 = d1.cpu().numpy().astype(np.uint64), d2.cpu().numpy().astype(np.uint64)
        # a chain stopped by the depth limit in the first call does nothing in the second
        assert ((d1 == split) | (d2 == 0)).all()
        done = d1 + d2
    np.testing.assert_array_equal(occ.cpu().numpy(), o_occ)
    np.testing.assert_array_equal(counts.cpu().numpy(), o_cnt)
    assert_stats_equal(hb.stats_to_numpy(stats), o_stats)
    np.testing.assert_array_equal(depth.cpu().numpy().astype(np.uint64), o_depth)
    np.testing.assert_array_equal(done, o_done)
    if split is None and log_cap:
        got = hb.log_to_numpy(log)
        for c in range(n_chains):
            n = min(int(o_stats["n_accept"][c]), log_cap)
            for f in ("step", "k", "a", "b"):
                np.testing.assert_array_equal(got[c][:n][f], o_log[c][:n][f])
    return o_stats, o_done


@pytest.mark.parametrize("select_best", [False, True])
@pytest.mark.parametrize("depth_limit", [0, 7, 150])
@pytest.mark.parametrize("team,threads", [(1, 64), (1, 512), (3, 128), (9, 512)])
def test_mc_run_ex_selection_and_depth(hb, select_best, depth_limit, team, threads):
    w = small("fcc", (4, 4, 4), [0.2, 0.2, 0.2, 0.4], 3, target_seed=5, K=24, n_steps=1500)
    st, done = run_both_ex(hb, w, 5, 1500, select_best, depth_limit,
                           opts={"mc_team": team, "mc_threads": threads, "mc_team_on": 256, "mc_team_off": 64})
    assert st["n_accept"].sum() > 50
    if depth_limit == 7:
        assert (done < 1500).all()                          # the depth limit stopped every chain early


@pytest.mark.parametrize("select_best", [False, True])
def test_mc_run_ex_split_run_carries_depth(hb, select_best):
    w = small("bcc", (5, 5, 5), [0.25] * 4, 3, K=32, n_steps=3000)
    run_both_ex(hb, w, 6, 3000, select_best, 400, split=1100, log_cap=0)


@pytest.mark.parametrize("lattice,dims,conc,S", LATTICES[:9])
def test_mc_run_ex_best_of_K_lattices(hb, lattice, dims, conc, S):
    w = small(lattice, dims, conc, S, target_seed=11, K=16)
    run_both_ex(hb, w, 3, 120, True, 0)


def test_mc_run_ex_c4_best_of_K_prefix_and_errors(hb):
    w = wl.config(4)
    st, _ = run_both_ex(hb, w, 4, 400, True, 0, log_cap=400)
    assert (st["n_accept"] > 300).all()
    h, _ = pair(hb, small("fcc", (3, 3, 3), [0.5, 0.5], 2))
    occ = h.init_random(2, seed=1)
    cnt, _, _ = h.sro_full(occ, want_alpha=False, want_obj=False)
    h.set_option("mc_engine", 1)
    with pytest.raises(hb.HeaError):                        # the window engine has no ex options
        h.mc_run_ex(occ, cnt, 10, 8, 1, select_best=True)


# ---- hea_pool_select (selection step of the global search) against the oracle's pool_select
@pytest.mark.parametrize("C,n_keep", [(12, 5), (9, 0), (7, 7), (300, 150)])
def test_pool_select_and_global_iterations(hb, C, n_keep):
    w = small("bcc", (4, 4, 4), [0.5, 0.25, 0.25], 2, target_seed=3, K=16)
    h, o = pair(hb, w)
    occ = h.init_random(C, seed=w.seed)
    counts, _, _ = h.sro_full(occ, want_alpha=False, want_obj=False)
    o_occ, o_cnt = occ.cpu().numpy().copy(), counts.cpu().numpy().copy()
    stats = h.new_stats(C)
    o_stats = ho.fresh_stats(C)
    for it in range(3):                                      # local search, then selection: three global iterations
        h.mc_run(occ, counts, 40, w.K, w.seed, step0=40 * it, stats=stats)
        o.mc_run(o_occ, o_cnt, 40, w.K, w.seed, step0=40 * it, stats=o_stats, eval_all=False, n_threads=8)
        if it == 0 and C >= 8:                               # an exact tie: two identical chains
            occ[C - 1], counts[C - 1], stats[C - 1] = occ[1].clone(), counts[1].clone(), stats[1].clone()
            o_occ[C - 1], o_cnt[C - 1], o_stats[C - 1] = o_occ[1], o_cnt[1], o_stats[1]
        order = h.pool_select(occ, counts, stats, n_keep, seed=1234 + it, new_chain0=10_000 * (it + 1))
        o_order = o.pool_select(o_occ, o_cnt, o_stats, n_keep, seed=1234 + it, new_chain0=10_000 * (it + 1))
        np.testing.assert_array_equal(order.cpu().numpy(), o_order)
        np.testing.assert_array_equal(occ.cpu().numpy(), o_occ)
        np.testing.assert_array_equal(counts.cpu().numpy(), o_cnt)
        assert_stats_equal(hb.stats_to_numpy(stats), o_stats)
        np.testing.assert_array_equal(hb.stats_to_numpy(stats)["last_accept_step"], o_stats["last_accept_step"])


# ---- full sizes, in the launch configuration of bench.py: every chain on the GPU, sampled chains through the oracle
def full_size_sampled(hb, w, n_steps, sample, threads=8):
    h, o = pair(hb, w)
    C = w.n_chains
    occ = h.init_random(C, seed=w.seed)
    counts, _, _ = h.sro_full(occ, want_alpha=False, want_obj=False)
    occ0 = occ.cpu().numpy().copy()
    stats, _ = h.mc_run(occ, counts, n_steps, w.K, w.seed)
    got = hb.stats_to_numpy(stats)
    occ_f, cnt_f = occ.cpu().numpy(), counts.cpu().numpy()
    # properties that hold at any size, on every chain
    for c in range(C):
        np.testing.assert_array_equal(np.bincount(occ_f[c], minlength=h.M), np.bincount(occ0[c], minlength=h.M))
    recount, _, obj = h.sro_full(occ)
    np.testing.assert_array_equal(recount.cpu().numpy(), cnt_f)                 # incremental == recount
    np.testing.assert_array_equal(obj.cpu().numpy(), got["J"])
    null_rate = got["n_null"].sum() / (C * n_steps * w.K)
    assert abs(null_rate - sum(x * x for x in w.conc) ** 2) < 2e-3             # (sum c_i^2)^2
    # sampled chains, element by element (chain c is independent of the batch it runs in)
    for c in sample:
        o_occ = o.init_random(1, w.seed, chain0=c)
        np.testing.assert_array_equal(o_occ[0], occ0[c])
        o_cnt = np.stack([o.pair_counts(o_occ[0])])
        o_st, _ = o.mc_run(o_occ, o_cnt, n_steps, w.K, w.seed, chain0=c, n_threads=1, eval_all=False)
        np.testing.assert_array_equal(occ_f[c], o_occ[0])
        np.testing.assert_array_equal(cnt_f[c], o_cnt[0])
        assert_stats_equal(got[c:c + 1], o_st)
    return got


def test_full_size_c2_all_chains_full_length(hb):
    w = wl.config(2)                                        # 1,024 chains x 100,000 steps x K=32
    full_size_sampled(hb, w, w.n_steps, sample=[0, 517, 1023])


def test_full_size_c3_all_chains(hb):
    w = wl.config(3)                                        # 256 chains x K=64; 200,000 of the 1e6 steps (oracle time)
    full_size_sampled(hb, w, 200_000, sample=[0, 255])


def test_full_size_c4_full_trajectory(hb):
    w = wl.config(4)                                        # 16 chains x 1e7 steps x K=128: the bench step
    h, o = pair(hb, w)
    got = full_size_sampled(hb, w, w.n_steps, sample=[])
    assert (got["n_accept"] > 60_000).all() and (got["J"] < 1e-8).all()
    # the same trajectory cut into two calls (different window and team schedules) gives the same moves
    occ = h.init_random(w.n_chains, seed=w.seed)
    counts, _, _ = h.sro_full(occ, want_alpha=False, want_obj=False)
    stats, _ = h.mc_run(occ, counts, 3_000_000, w.K, w.seed)
    h.mc_run(occ, counts, 7_000_000, w.K, w.seed, step0=3_000_000, stats=stats)
    st2 = hb.stats_to_numpy(stats)
    for f in ("n_accept", "n_null", "hash", "last_accept_step", "J"):
        np.testing.assert_array_equal(got[f], st2[f])
    # one sampled chain against the oracle over the first 1,000,000 steps (accept regime, transition, 930,000 reject steps)
    o_occ = o.init_random(1, w.seed, chain0=11)
    o_cnt = np.stack([o.pair_counts(o_occ[0])])
    o_st, _ = o.mc_run(o_occ, o_cnt, 1_000_000, w.K, w.seed, chain0=11, n_threads=1, eval_all=False)
    occ = h.init_random(w.n_chains, seed=w.seed)
    counts, _, _ = h.sro_full(occ, want_alpha=False, want_obj=False)
    stats, _ = h.mc_run(occ, counts, 1_000_000, w.K, w.seed)
    assert_stats_equal(hb.stats_to_numpy(stats)[11:12], o_st)
    np.testing.assert_array_equal(occ.cpu().numpy()[11], o_occ[0])
