"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element,
on the same seeded inputs.  Bar (BASELINE.json north_star): accept/reject sequences and vertex
configurations BIT-EXACT; N within relative Frobenius error 1e-10 in FP64."""
import numpy as np
import pytest

from ctaux_workloads import get_config, table_for, walker_seeds
from oracle.ctaux_oracle import T0, T1, OracleWalker, philox

from parity_helpers import (compare_configs, compare_logs, compare_N, frob_rel, full_parity, load_thermalised,
                            parity_from_state, run_oracle)

# N is held to 1e-10 in EVERY case below, thermalising or not, with or without a periodic rebuild: the library's error
# monitor (ctaux_params.n_tol, default 1e-10) estimates the forward error of N on the device and rebuilds when needed.

pytestmark = pytest.mark.gpu


def _pkg():
    import paper_1901_01047_b200 as pkg
    return pkg


def test_P12_device_philox_equals_oracle_philox():
    rng = np.random.default_rng(0)
    ctr = rng.integers(0, 2 ** 32, size=(257, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2 ** 32, size=(257, 2), dtype=np.uint64).astype(np.uint32)
    ctr[0] = 0
    key[0] = 0
    ctr[1] = [5, 0, 1, 1]
    dev = _pkg().debug_philox(ctr, key)
    for i in range(ctr.shape[0]):
        assert dev[i].tolist() == philox(ctr[i], key[i]).tolist()


@pytest.mark.parametrize("b_nmajor", [0, 1])
@pytest.mark.parametrize("M,N,K,alpha,beta", [(1, 1, 1, -1.5, 0.5), (8, 8, 4, -1.5, 0.5), (130, 70, 33, -1.5, 0.5),
                                              (128, 128, 64, -1.0, 1.0), (257, 511, 100, -1.5, 0.5),
                                              (1000, 40, 1000, 1.0, 0.0), (64, 1000, 7, -1.0, 1.0),
                                              (300, 300, 5, 2.0, 0.5), (1900, 1834, 64, -1.0, 1.0),
                                              (64, 1834, 1834, 1.0, 0.0), (1898, 64, 1898, 1.0, 0.0),
                                              (700, 900, 129, 1.0, 1.0)])
def test_dgemm_tiles_against_torch_fp64(M, N, K, alpha, beta, b_nmajor):
    """The TMA-staged DMMA GEMM tile with both right-operand layouts the walker uses (K-major: N in the candidate-row
    product and the LU panels; N-major: V in the flush, g_ext in the candidate-column product): several tiles,
    several K chunks, ragged tails in M, N and K, the in-place C0 - A*B form, against torch's FP64 matmul."""
    import torch
    pkg = _pkg()
    g = torch.Generator(device="cpu").manual_seed(M * 7 + N * 3 + K)
    rnd = lambda r, c: torch.randn(r, c, generator=g, dtype=torch.float64)
    A = pkg.colmajor(M, K, fill=rnd)
    B = pkg.colmajor(K, N, fill=rnd)
    C0 = pkg.colmajor(M, N, fill=rnd)
    C = pkg.colmajor(M, N)
    C.copy_(C0)
    out = pkg.ctaux_dgemm(A, B, C, alpha=alpha, beta=beta, b_nmajor=b_nmajor)
    ref = beta * C0 + alpha * (A @ B)
    torch.cuda.synchronize()
    scale = float(ref.abs().max()) + 1e-300
    assert float((out - ref).abs().max()) / scale < 1e-13 * max(K, 1)


@pytest.mark.parametrize("ci,nw", [(0, 1), (1, 5), (2, 3)])
def test_reset_builds_inverse(ci, nw):
    """S1 + S5: N after reset equals the oracle's direct inverse of A built from the same vertices."""
    cfg = get_config(ci)
    table = table_for(cfg)
    W = _pkg().Walkers.from_config(cfg, table, n_walkers=nw)
    seeds = walker_seeds(nw, first=10)
    W.reset(seeds)
    for w in range(nw):
        o = OracleWalker.from_config(cfg, table, int(seeds[w]), T0)
        o.reset(cfg["init_k"])
        compare_configs(W.get_config(w), o.config(), f"reset walker {w}")
        compare_N(W, w, o, f"reset walker {w}")
        assert W.get_stats(w)["sign"] == o.sign
        # P7 on the device matrix itself: A N = 1.  A's columns carry the factors E_j (up to e^gamma),
        # so the residual is taken on the column-equilibrated matrix A D^-1 (D N is its inverse).
        for s in range(2):
            k = o.k
            A = o.A(s)
            dcol = np.abs(A).max(axis=0)
            res = (A / dcol) @ (dcol[:, None] * W.get_N(w, s)) - np.eye(k)
            assert np.linalg.norm(res) / np.sqrt(k) < 1e-10


# fused = 1: the single-kernel small-k path (walker_fused.cuh, what configs 1-2 run by default);
# fused = -1: the delayed-block path (S2 GEMMs, S3 over the Gamma block, S4 flush) the large configs run.
def test_rebuild_large_k_kernels_at_small_size():
    """max_k > 512 selects the large-k kernels (64x64 4-warp GEMM tiles, split-K, the 8-CTA cluster LU panel):
    S1 + S5 and a few sweeps against the oracle on config 3 with the capacity raised to 600."""
    cfg = dict(get_config(2), max_k=600)
    full_parity(cfg, 3, 10, T1)           # ends on a rebuild: N fresh from the cluster LU
    W, orcs, worst = full_parity(cfg, 2, 0, T0)   # reset only: direct inverse of the random start
    assert worst < 1e-10


@pytest.mark.parametrize("fused", [1, -1])
def test_config1_full_lockstep_T0(fused):
    """Config 1 in full (200 warm-up + 1000 sweeps, 1 walker, delay 8) against brute force T0."""
    cfg = get_config(0)
    W, orcs, worst = full_parity(cfg, 1, cfg["warmup_sweeps"] + cfg["sweeps"], T0, fused=fused)
    st = W.get_stats(0)
    assert st["rebuilds"] - st["monitor_rebuilds"] == 120


@pytest.mark.parametrize("fused", [1, -1])
def test_config2_batched_walkers_T0_prefix_and_T1(fused):
    cfg = get_config(1)
    full_parity(cfg, 16, 12, T0, fused=fused)          # brute force on a prefix, 16 walkers
    full_parity(cfg, 256, 40, T1, fused=fused)         # all 256 walkers, rank-1 oracle


def test_config2_fused_without_rebuild_N_1e10():
    """The fused path's incrementally updated N (rank-1 updates in shared memory, no rebuild) from the
    equilibrated state of an oracle chain: 32 walkers x 15 sweeps."""
    cfg = get_config(1)
    table = table_for(cfg)
    o = OracleWalker.from_config(cfg, table, 0, T1)
    o.reset(cfg["init_k"])
    o.sweep(60)
    parity_from_state(cfg, (o.config(), o.next_id, o.p), walker_seeds(32), 15, T1, fused_small=1)


def test_config3_T1():
    cfg = get_config(2)
    full_parity(cfg, 64, 6, T1)
    full_parity(cfg, 64, 10, T1)          # ends on the config's rebuild cadence: N fresh from S5
    full_parity(cfg, 2, 1, T0)


def test_config3_thermalised_start_N_1e10():
    """Config 3 from the oracle-thermalised configuration (40 sweeps), 16 seeds, 8 sweeps WITHOUT any
    rebuild on the device: the incrementally updated N (about 65 flushes of rank <= 32) within 1e-10."""
    cfg = get_config(2)
    W, orcs, worst = parity_from_state(cfg, load_thermalised(cfg["name"]), walker_seeds(16), 8, T1)
    assert sum(W.get_stats(w)["flushes"] for w in range(16)) > 500


# delay 128 / 256: the two-CTA cluster form of the S3 kernel (S^-1 of one spin per CTA in shared memory / in L2)
@pytest.mark.parametrize("delay,rebuild,cand", [(1, 0, 0), (8, 0, 3), (64, 3, 0), (16, 1, 40), (128, 0, 0), (256, 0, 0),
                                                (100, 0, 0)])
def test_chain_independent_of_delay_rebuild_window(delay, rebuild, cand):
    """Q18-Q20: delay, rebuild cadence and the candidate window are performance knobs only."""
    cfg = get_config(1)
    full_parity(cfg, 4, 10, T1, delay=delay, rebuild_every=rebuild, cand_window=cand, fused=-1)


@pytest.mark.parametrize("fused", [1, -1])
def test_sweep_calls_continue_the_chain(fused):
    cfg = get_config(1)
    table = table_for(cfg)
    pkg = _pkg()
    seeds = walker_seeds(3, first=100)
    a = pkg.Walkers.from_config(cfg, table, n_walkers=3, log_capacity=4000, fused_small=fused)
    a.reset(seeds)
    for n in (1, 2, 3):
        a.sweep(n)
    b = pkg.Walkers.from_config(cfg, table, n_walkers=3, log_capacity=4000, fused_small=fused)
    b.reset(seeds)
    b.sweep(6)
    for w in range(3):
        # block boundaries differ (a block ends with each sweep call), so R agrees to rounding only
        compare_logs(a.get_log(w), b.get_log(w), f"split sweeps walker {w}")
        compare_configs(a.get_config(w), b.get_config(w))
        assert a.get_stats(w)["proposals"] == b.get_stats(w)["proposals"]


@pytest.mark.parametrize("fused", [1, -1])
def test_empty_start_and_tiny_cluster_edge_cases(fused):
    """Degenerate cases: empty initial configuration (removals on k=0 are rejected), 1x1 cluster."""
    cfg = get_config(0)
    full_parity(cfg, 3, 30, T0, init_k=0, fused=fused)
    atom = dict(cfg, name="atom", Lx=1, Ly=1, mu=0.0)
    full_parity(atom, 2, 30, T0, init_k=0, fused=fused)


@pytest.mark.parametrize("fused", [1, -1])
def test_set_state_resumes_an_oracle_chain(fused):
    """ctaux_set_state: continue on the device from a configuration produced by the oracle."""
    cfg = get_config(1)
    table = table_for(cfg)
    o = OracleWalker.from_config(cfg, table, 9, T1)
    o.reset(cfg["init_k"])
    o.sweep(5)
    c0, nid, p0 = o.config(), o.next_id, o.p
    o.clear_log()
    o.sweep(4)
    W = _pkg().Walkers.from_config(cfg, table, n_walkers=1, log_capacity=2000, fused_small=fused)
    W.set_state([9], [c0], [nid], [p0])
    W.sweep(4)
    compare_logs(W.get_log(0), o.log(), "resumed")
    compare_configs(W.get_config(0), o.config(), "resumed")
    compare_N(W, 0, o, "resumed")


@pytest.mark.parametrize("fused", [1, -1])
def test_capacity_error_is_loud(fused):
    cfg = get_config(1)
    table = table_for(cfg)
    pkg = _pkg()
    W = pkg.Walkers(cfg["Lx"], cfg["Ly"], cfg["beta"], cfg["U"], cfg["K"], table, delay=8, n_walkers=2,
                    init_k=5, max_k=12, fused_small=fused)
    W.reset(walker_seeds(2))
    with pytest.raises(pkg.CtauxError) as ei:
        W.sweep(50)
    assert ei.value.code == -2


def test_fused_path_spills_to_the_delayed_path():
    """2x2 cluster at beta = 18: <k> ~ 110 sits at the shared-memory capacity of the fused kernel (116 slots
    for max_k = 150), so walkers keep crossing it: they spill to the delayed-block path mid-sweep and come
    back at the next call.  Same chain, bit for bit."""
    cfg = dict(get_config(1), name="cfg2_beta18", beta=18.0, max_k=150, init_k=74, rebuild_every=4)
    W, orcs, worst = full_parity(cfg, 8, 16, T1, fused=1)
    st = [W.get_stats(w) for w in range(8)]
    assert sum(x["flushes"] for x in st) > 0, "no walker ever spilled: the test does not reach the capacity"
    assert max(o.k for o in orcs) > 100


def test_fused_path_refuses_what_does_not_fit():
    cfg = get_config(2)                      # max_k 384: 2 x 384^2 x 8 B does not fit one SM
    pkg = _pkg()
    with pytest.raises(pkg.CtauxError) as ei:
        pkg.Walkers.from_config(cfg, table_for(cfg), n_walkers=1, fused_small=1)
    assert ei.value.code == -2


@pytest.mark.slow
def test_config4_prefix_T1():
    """Config 4 (6x6, beta 20) from reset, k ~ 1100-1300: first 2 sweeps of 2 walkers against T1."""
    cfg = get_config(3)
    full_parity(cfg, 2, 2, T1)


@pytest.mark.slow
def test_config4_growth_from_empty_start_outruns_the_grid_hint():
    """Large-k path (max_k > 512) from the EMPTY configuration without any rebuild: k grows from 0 to ~1000 in 18
    sweeps, by up to ~60 per block step, i.e. several hundred between two polls of the host's live-order hint, so the
    flush grid sized from that hint is too small again and again; the kernel strides over the tiles the grid does
    not cover.  Any row or column of N left unwritten would derail the decisions within a few proposals."""
    cfg = get_config(3)
    W, orcs, worst = full_parity(cfg, 2, 18, T1, init_k=0, rebuild_every=0, check_N=False)
    assert min(o.k for o in orcs) > 800
    W.rebuild()
    for w, o in enumerate(orcs):
        compare_N(W, w, o, f"config 4 after growth + rebuild, walker {w}")


@pytest.mark.slow
def test_config4_thermalised_start_N_1e10():
    """Config 4 at its full size (k ~ 1720, delay 64, the launch configuration bench.py times) from the
    oracle-thermalised configuration: 4 seeds x 1 sweep without rebuild, logs bit-exact, N within 1e-10."""
    cfg = get_config(3)
    parity_from_state(cfg, load_thermalised(cfg["name"]), walker_seeds(4), 1, T1)


@pytest.mark.slow
@pytest.mark.parametrize("delay", [128, 256])
def test_config4_thermalised_start_cluster_kernel(delay):
    """Same start, delay 128 / 256 (config 5's delays): the S3 kernel runs as a two-CTA cluster per walker."""
    cfg = get_config(3)
    W, orcs, worst = parity_from_state(cfg, load_thermalised(cfg["name"]), walker_seeds(2), 1, T1, delay=delay)
    assert max(W.get_stats(w)["sum_rank"] / max(W.get_stats(w)["flushes"], 1) for w in range(2)) > 0.5 * delay


@pytest.mark.parametrize("ci,modes,nw,sweeps", [(2, (0, -1), 4, 6), (3, (1, -1), 2, 12)])
def test_cuda_graph_path_runs_the_same_chain(ci, modes, nw, sweeps):
    """ctaux_params.graph_mode: a poll interval of block steps relaunched as a CUDA graph (default for max_k <= 512, on
    request for every size) against plain launches, device against device; the large configuration starts EMPTY, so that
    its live order crosses several of the grid size classes a graph is captured for.
    Same kernels, same arithmetic per tile: decisions, configurations and counters identical; on the large configuration
    the split-K factor of the S2 products follows the grid size, so logged ratios and N agree to rounding only."""
    pkg = _pkg()
    cfg = get_config(ci)
    table = table_for(cfg)
    seeds = walker_seeds(nw, first=21)
    runs = []
    for mode in modes:
        W = pkg.Walkers.from_config(cfg, table, n_walkers=nw, init_k=0 if ci == 3 else cfg["init_k"], graph_mode=mode, fused_small=-1,
                                    log_capacity=sweeps * cfg["max_k"], rebuild_every=3)
        W.reset(seeds)
        W.sweep(2)
        W.sweep(sweeps - 2)
        runs.append(W)
    A, B = runs
    for w in range(nw):
        what = f"{cfg['name']} graph_mode {modes[0]} vs {modes[1]}, walker {w}"
        compare_logs(A.get_log(w), B.get_log(w), what)
        compare_configs(A.get_config(w), B.get_config(w), what)
        sa, sb = A.get_stats(w), B.get_stats(w)
        for f in ("k", "proposals", "next_id", "sign", "acc_ins", "acc_rem", "sweeps", "blocks", "flushes"):
            assert sa[f] == sb[f], (what, f)
        assert sa["k"] > 150      # (the large configuration has crossed at least two grid size classes of 128 by then)
        for sp in range(2):
            Na, Nb = A.get_N(w, sp), B.get_N(w, sp)
            assert np.linalg.norm(Na - Nb) <= 1e-10 * np.linalg.norm(Nb), what
    if ci == 2:      # same grids, same split: the graph path counts exactly what it launches
        assert A._L.ctaux_launch_count(A._h) == B._L.ctaux_launch_count(B._h)
    A.close(); B.close()


def test_error_codes_through_the_abi():
    """Calls that are not valid fail with their CTAUX_E* code and leave the process alive."""
    pkg = _pkg()
    cfg = get_config(0)
    table = table_for(cfg)
    W = pkg.Walkers.from_config(cfg, table)
    with pytest.raises(pkg.CtauxError) as ei:
        W.sweep(1)                       # sweep before reset
    assert ei.value.code == -5
    with pytest.raises(pkg.CtauxError) as ei:
        W.rebuild()
    assert ei.value.code == -5
    W.reset([3])
    W.sweep(2)
    L = pkg.load_library()
    import ctypes as C
    k = C.c_int32(0)
    assert L.ctaux_get_config(W._h, 5, C.byref(k), None, None, None, None, 0) == -1      # walker out of range
    assert L.ctaux_get_config(W._h, 0, C.byref(k), None, None, None, None, 0) == 0 and k.value == W.get_stats(0)["k"]
    buf = np.zeros(4, np.int32)
    assert L.ctaux_get_config(W._h, 0, C.byref(k), None, buf.ctypes.data, None, None, 1) == (-2 if k.value > 1 else 0)
    assert L.ctaux_get_N(W._h, 0, 2, buf.ctypes.data, 64) == -1                             # spin out of range
    assert L.ctaux_get_N(W._h, 0, 0, buf.ctypes.data, 0) == (-1 if k.value > 0 else 0)      # ld < k
    W.close()
    with pytest.raises(pkg.CtauxError) as ei:   # invalid parameters are refused before anything is allocated
        pkg.Walkers(2, 2, 2.0, 4.0, 1.0, table, delay=300, n_walkers=1, init_k=1, max_k=64)
    assert ei.value.code == -1


@pytest.mark.parametrize("nw", [5, 20])
def test_batched_readout_equals_per_walker_readout(nw):
    """nw = 20 takes the packed path of ctaux_get_N_all (device-side pack into the host layout, one 2-D copy)."""
    pkg = _pkg()
    cfg = get_config(1)
    W = pkg.Walkers.from_config(cfg, table_for(cfg), n_walkers=nw)
    W.reset(walker_seeds(nw, first=7))
    W.sweep(3)
    cfgs = W.get_config_all()
    Ns = W.get_N_all([len(c["site"]) for c in cfgs])
    for w in range(nw):
        one = W.get_config(w)
        for f in one:
            assert one[f].tobytes() == cfgs[w][f].tobytes()
        for s in range(2):
            assert np.array_equal(W.get_N(w, s), Ns[w][s])
    W.close()


def test_packed_state_round_trip_continues_the_chain():
    """The C ABI's batched forms as the bench's end-to-end leg uses them: get_state_packed (pinned host buffers) ->
    set_state_packed on a second context -> both continue; identical configurations, counters and N afterwards, and
    the packed N equals the per-walker getter."""
    pkg = _pkg()
    cfg = get_config(1)
    table = table_for(cfg)
    nw = 18
    seeds = walker_seeds(nw, first=3)
    A = pkg.WalkerGroups(2, nw, lambda g, nb, stream: pkg.Walkers.from_config(cfg, table, n_walkers=nb, stream=stream))
    A.reset(seeds)
    A.sweep(4)
    st = A.get_state_packed(with_N=True)
    mk = cfg["max_k"]
    for g, s_ in enumerate(st):
        for i in range(A.per):
            k = int(s_["k"][i])
            for sp in range(2):
                blk = s_["N"][(2 * i + sp) * mk * mk:(2 * i + sp) * mk * mk + k * k].reshape((k, k), order="F")
                assert np.array_equal(blk, A.get_N(g * A.per + i, sp))
    B = pkg.WalkerGroups(2, nw, lambda g, nb, stream: pkg.Walkers.from_config(cfg, table, n_walkers=nb, stream=stream))
    B.set_state_packed(seeds, st)
    A.sweep(3)
    B.sweep(3)
    for w in range(nw):
        ca, cb = A.get_config(w), B.get_config(w)
        for f in ca:
            assert ca[f].tobytes() == cb[f].tobytes()
        sa, sb = A.get_stats(w), B.get_stats(w)
        assert sa["proposals"] == sb["proposals"] and sa["next_id"] == sb["next_id"] and sa["sign"] == sb["sign"]
        for sp in range(2):
            Na, Nb = A.get_N(w, sp), B.get_N(w, sp)
            assert np.linalg.norm(Na - Nb) <= 1e-10 * np.linalg.norm(Na)
    A.close(); B.close()


@pytest.mark.parametrize("fused", [1, -1])
def test_walker_groups_run_the_same_chains(fused):
    """WalkerGroups (walkers split over contexts / streams / host threads) against one context: identical
    configurations, counters and N for every walker; batched fetch_all equals the per-walker getters."""
    pkg = _pkg()
    cfg = get_config(1)
    table = table_for(cfg)
    B, G, ns = 6, 3, 7
    seeds = walker_seeds(B, first=40)
    one = pkg.Walkers.from_config(cfg, table, n_walkers=B, fused_small=fused)
    one.reset(seeds)
    one.sweep(ns)
    grp = pkg.WalkerGroups(G, B, lambda g, nb, stream: pkg.Walkers.from_config(cfg, table, n_walkers=nb, stream=stream,
                                                                                 fused_small=fused))
    grp.reset(seeds)
    grp.sweep(3)
    grp.sweep(ns - 3)
    cfgs, stats, Ns = grp.fetch_all()
    for w in range(B):
        compare_configs(cfgs[w], one.get_config(w), f"group walker {w}")
        s1 = one.get_stats(w)
        for f in ("k", "proposals", "next_id", "sign", "acc_ins", "acc_rem", "sweeps"):
            assert stats[w][f] == s1[f], (w, f)
        for s in range(2):
            assert frob_rel(Ns[w][s], one.get_N(w, s)) < 1e-10
            assert np.array_equal(Ns[w][s], grp.get_N(w, s))
    grp.close()
    one.close()


@pytest.mark.parametrize("fused", [1, -1])
def test_newton_schulz_refresh_config2(fused):
    """rebuild_mode 1: the periodic rebuild is one Newton-Schulz step N <- N (2 - A N) (two GEMMs) instead of the
    LU.  Same chain; N right after a refresh within 1e-10 of the oracle's direct inverse."""
    cfg = get_config(1)
    W, orcs, worst = full_parity(cfg, 16, 20, T1, fused=fused, rebuild_mode=1, rebuild_every=5)
    assert all(W.get_stats(w)["rebuilds"] - W.get_stats(w)["monitor_rebuilds"] == 4 for w in range(16))
    full_parity(cfg, 4, 12, T0, fused=fused, rebuild_mode=1, rebuild_every=1)


def test_newton_schulz_refresh_config3_and_large_k_kernels():
    cfg = get_config(2)
    full_parity(cfg, 8, 10, T1, rebuild_mode=1, rebuild_every=5, n_tol=1e-10)
    big = dict(cfg, max_k=600)
    full_parity(big, 2, 6, T1, rebuild_mode=1, rebuild_every=3)


@pytest.mark.slow
def test_newton_schulz_refresh_config4_thermalised():
    """Config 4 at full size from the thermalised start: 2 sweeps with a refresh after each; the refreshed N
    against the oracle's from-scratch inverse."""
    cfg = get_config(3)
    W, orcs, worst = parity_from_state(cfg, load_thermalised(cfg["name"]), walker_seeds(2), 2, T1,
                                       rebuild_every=1, rebuild_mode=1)
    assert all(W.get_stats(w)["rebuilds"] - W.get_stats(w)["monitor_rebuilds"] == 2 for w in range(2))


# ---------------------------------------------------------------- NEXT-1: auxiliary-spin flips (flip_moves = 1)
@pytest.mark.parametrize("fused", [1, -1])
def test_flips_config1_and_2(fused):
    """Three-move chain (insert / remove / flip) against the oracle: brute force on config 1 and a config-2
    prefix, rank-1 oracle on 64 walkers; logs, configurations (spins!), counters bit-exact, N within 1e-10."""
    cfg = get_config(0)
    W, orcs, worst = full_parity(cfg, 1, 300, T0, fused=fused, flips=1)
    assert W.get_stats(0)["acc_flip"] > 50
    cfg = get_config(1)
    full_parity(cfg, 8, 12, T0, fused=fused, flips=1)
    full_parity(cfg, 64, 40, T1, fused=fused, flips=1)


@pytest.mark.parametrize("delay", [1, 16, 64, 128])
def test_flips_chain_independent_of_delay(delay):
    cfg = get_config(1)
    full_parity(cfg, 4, 10, T1, delay=delay, rebuild_every=0, fused=-1, flips=1)


def test_flips_config3_thermalised():
    cfg = get_config(2)
    W, orcs, worst = parity_from_state(cfg, load_thermalised(cfg["name"]), walker_seeds(8), 6, T1, flips=1)
    assert sum(W.get_stats(w)["acc_flip"] for w in range(8)) > 100


@pytest.mark.slow
def test_flips_config4_thermalised():
    cfg = get_config(3)
    W, orcs, worst = parity_from_state(cfg, load_thermalised(cfg["name"]), walker_seeds(2), 1, T1, flips=1)
    assert sum(W.get_stats(w)["acc_flip"] for w in range(2)) > 50


def test_numerical_guard_is_chain_neutral():
    """guard_amp only moves block boundaries: off, default and an aggressive setting give the same decisions;
    the aggressive one ends many more blocks early."""
    pkg = _pkg()
    cfg = get_config(1)
    table = table_for(cfg)
    seeds = walker_seeds(6, first=200)
    logs, ends = [], []
    for ga in (-1.0, 0.0, 5.0):
        W = pkg.Walkers.from_config(cfg, table, n_walkers=6, fused_small=-1, rebuild_every=0, log_capacity=3000, guard_amp=ga)
        W.reset(seeds)
        W.sweep(12)
        logs.append([W.get_log(w) for w in range(6)])
        ends.append(sum(W.get_stats(w)["guard_ends"] for w in range(6)))
        W.close()
    for w in range(6):
        for other in (1, 2):
            for f in ("p", "type", "arg", "tau", "spin", "accepted", "u"):
                assert logs[0][w][f].tobytes() == logs[other][w][f].tobytes(), (w, other, f)
    assert ends[0] == 0 and ends[2] > ends[1] >= 0 and ends[2] > 20


def test_error_monitor_estimate_tracks_the_true_error_and_is_chain_neutral():
    """ctaux_params.n_tol: (a) with the trigger out of reach (n_tol = 1e300) the monitor only measures: its estimate
    of |N - A^-1|_F / |N|_F after 6 un-rebuilt sweeps from the random start of config 3 (A nearly singular there, the
    drift is large) agrees with the true error against the oracle's direct inverse within the spread of a 4-probe
    Hutchinson estimate; (b) with the monitor off the same chains drift beyond the bar, with the default n_tol they are
    held to 1e-10; (c) the decisions are identical in all three runs."""
    pkg = _pkg()
    cfg = get_config(2)
    table = table_for(cfg)
    nw, ns = 64, 6
    seeds = walker_seeds(nw)
    orcs = run_oracle(cfg, table, seeds, ns, T1)
    logs, drift = {}, {}
    for tag, tol in (("measure", 1e300), ("off", -1.0), ("on", 0.0)):
        W = pkg.Walkers.from_config(cfg, table, n_walkers=nw, rebuild_every=0, log_capacity=3000, n_tol=tol)
        W.reset(seeds)
        W.sweep(ns)
        logs[tag] = [W.get_log(w) for w in range(nw)]
        true = [max(frob_rel(W.get_N(w, s), orcs[w].N(s)) for s in range(2)) for w in range(nw)]
        drift[tag] = max(true)
        st = [W.get_stats(w) for w in range(nw)]
        if tag == "measure":
            assert all(x["monitor_rebuilds"] == 0 for x in st)
            # (walkers whose drift is at the level of the oracle's own inverse, ~1e-12, say nothing about the estimator)
            ratio = np.array([x["err_est"] / t for x, t in zip(st, true) if t > 5e-12])
            assert ratio.size >= 8 and 0.2 < np.median(ratio) < 5.0 and ratio.min() > 0.03 and ratio.max() < 30.0, ratio
        if tag == "off":
            assert all(x["monitor_rebuilds"] == 0 and x["err_est"] == 0.0 for x in st)
        if tag == "on":
            assert sum(x["monitor_rebuilds"] for x in st) > 0
        W.close()
    assert drift["off"] > 1e-10 and drift["measure"] > 1e-10, "the case does not drift: it does not test the monitor"
    assert drift["on"] < 1e-10
    for w in range(nw):
        for f in ("p", "type", "arg", "tau", "spin", "accepted", "u"):
            assert logs["off"][w][f].tobytes() == logs["on"][w][f].tobytes() == logs["measure"][w][f].tobytes()
        compare_logs(logs["on"][w], orcs[w].log(), f"monitor on, walker {w}")


@pytest.mark.parametrize("flips", [0, 1])
def test_P6_atomic_limit_mean_order_on_the_device(flips):
    """Pin P6 evaluated on the DEVICE chain itself (no oracle log involved): Nc = 1, xi = 0,
    <k> = K + (beta U/2)/(1 + e^{-beta U/2}) = 4.92806, from sum_k / proposals over 128 chains."""
    import math
    from ctaux_workloads import atomic_limit_table
    pkg = _pkg()
    beta, U, K = 2.0, 4.0, 1.0
    want = K + (beta * U / 2) / (1 + math.exp(-beta * U / 2))
    nw = 128
    W = pkg.Walkers(1, 1, beta, U, K, atomic_limit_table(64), delay=8, n_walkers=nw, init_k=5, max_k=64,
                    rebuild_every=50, flip_moves=flips)
    W.reset(walker_seeds(nw, first=1000))
    W.sweep(300)                                   # thermalise
    a = [W.get_stats(w) for w in range(nw)]
    W.sweep(3000)
    b = [W.get_stats(w) for w in range(nw)]
    means = np.array([(y["sum_k"] - x["sum_k"]) / (y["proposals"] - x["proposals"]) for x, y in zip(a, b)])
    err = means.std(ddof=1) / math.sqrt(nw)
    assert abs(means.mean() - want) < max(4 * err, 0.01), (means.mean(), err, want)
    W.close()


def test_P5_U_zero_on_the_device():
    """Degenerate case gamma = 0 (BASELINE.json: "gamma -> 0 leaves N = 1"): the chain is the birth-death process with
    R_ins = K/(k+1), R_rem = k/K, stationary k ~ Poisson(K): mean = variance = K on the device chains; N = 1; bit-exact
    against the oracle; the delayed-block path (which divides by E - 1) refuses U = 0 loudly."""
    pkg = _pkg()
    K = 1.5
    cfg = dict(get_config(0), name="U0", U=0.0, K=K, init_k=3)
    full_parity(cfg, 4, 50, T1, fused=1)
    table = table_for(cfg)
    nw = 256
    W = pkg.Walkers(2, 2, cfg["beta"], 0.0, K, table, delay=8, n_walkers=nw, init_k=3, max_k=64, rebuild_every=0)
    W.reset(walker_seeds(nw, first=500))
    W.sweep(50)
    ks = []
    for rep in range(40):
        W.sweep(3)
        ks += [W.get_stats(w)["k"] for w in range(nw)]
    ks = np.array(ks, dtype=np.float64)
    n = ks.size
    assert abs(ks.mean() - K) < 5 * np.sqrt(K / n) * 3       # autocorrelated samples: generous factor
    assert abs(ks.var() - K) < 0.15
    k0 = W.get_stats(0)["k"]
    assert np.array_equal(W.get_N(0, 0), np.eye(k0)) and np.array_equal(W.get_N(0, 1), np.eye(k0))
    W.close()
    with pytest.raises(pkg.CtauxError) as ei:
        pkg.Walkers(2, 2, cfg["beta"], 0.0, K, table, delay=8, n_walkers=1, init_k=3, max_k=64, fused_small=-1)
    assert ei.value.code == -1


@pytest.mark.slow
def test_config5_thermalised_start_full_size_delay_128_and_256():
    """Config 5 at full size (6x6, beta 40, k ~ 3600; split-K S2 GEMMs, rank-128 / rank-256 flushes; S3 as a 2-CTA
    cluster per walker with S^-1 in shared memory at delay 128 and in L2 at delay 256 -- the two launch
    configurations bench.py times).  Two walkers, each from the thermalised configuration of its OWN oracle seed
    (tests/golden/thermalised_cfg5_6x6_b40_seed{0,1}.txt, >= 25 oracle sweeps): 1600 proposals (ctaux_propose; 3-4
    blocks at delay 256, 6-7 at delay 128) against T1, decisions bit-exact, N within 1e-10.  The oracle runs once (its
    chain does not depend on the delay); a whole sweep at this size costs the plain-C++ oracle ~5 min."""
    from concurrent.futures import ThreadPoolExecutor
    cfg = get_config(4)
    table = table_for(cfg)
    states = [load_thermalised(cfg["name"], sd) for sd in (0, 1)]
    seeds = walker_seeds(2)
    nprop = 1600

    def one(i):
        c0, next_id, p0 = states[i]
        o = OracleWalker.from_config(cfg, table, int(seeds[i]), T1)
        o.set_state(c0["site"], c0["tau"], c0["spin"], c0["id"], next_id, p0)
        o.propose(nprop)
        return o

    with ThreadPoolExecutor(max_workers=2) as ex:
        fut = [ex.submit(one, i) for i in range(2)]
        Ws = []
        for delay in (128, 256):
            W = _pkg().Walkers(cfg["Lx"], cfg["Ly"], cfg["beta"], cfg["U"], cfg["K"], table, delay=delay, n_walkers=2,
                               init_k=0, max_k=cfg["max_k"], rebuild_every=0, log_capacity=nprop + 64)
            W.set_state(seeds, [s[0] for s in states], [s[1] for s in states], [s[2] for s in states])
            W.propose(nprop)
            Ws.append((delay, W))
        orcs = [f.result() for f in fut]
    for delay, W in Ws:
        for w, o in enumerate(orcs):
            what = f"config 5 delay {delay} walker {w}"
            compare_logs(W.get_log(w), o.log(), what)
            compare_configs(W.get_config(w), o.config(), what)
            st = W.get_stats(w)
            assert st["k"] == o.k and st["proposals"] == o.p and st["next_id"] == o.next_id and st["sign"] == o.sign, what
            assert st["proposals"] == states[w][2] + nprop
            assert st["flushes"] >= 3 and st["sum_rank"] / st["flushes"] > 0.5 * delay
            compare_N(W, w, o, what)
        W.close()


@pytest.mark.parametrize("fused", [1, -1])
def test_propose_calls_split_the_chain_anywhere(fused):
    """ctaux_propose (a partial sweep of exactly n proposals) mixed with ctaux_sweep: the chain depends on the proposal
    counter only.  Config 2 (fused small-k kernel and delayed path) in lock step with the oracle's propose / sweep."""
    pkg = _pkg()
    cfg = get_config(1)
    table = table_for(cfg)
    nw = 3
    seeds = walker_seeds(nw, first=11)
    W = pkg.Walkers.from_config(cfg, table, n_walkers=nw, fused_small=fused, log_capacity=4000, rebuild_every=2)
    W.reset(seeds)
    orcs = []
    for sd in seeds:
        o = OracleWalker.from_config(cfg, table, int(sd), T1)
        o.reset(cfg["init_k"])
        orcs.append(o)
    for kind, n in (("p", 37), ("s", 1), ("p", 1), ("p", 150), ("s", 2), ("p", 5)):
        if kind == "p":
            W.propose(n)
            [o.propose(n) for o in orcs]
        else:
            W.sweep(n)
            [o.sweep(n) for o in orcs]
        for w, o in enumerate(orcs):
            st = W.get_stats(w)
            assert st["proposals"] == o.p and st["k"] == o.k, (kind, n, w)
    for w, o in enumerate(orcs):
        what = f"propose/sweep mix, fused {fused}, walker {w}"
        compare_logs(W.get_log(w), o.log(), what)
        compare_configs(W.get_config(w), o.config(), what)
        compare_N(W, w, o, what)
    assert W._L.ctaux_propose(W._h, -1) == -1
    W.propose(0)
    W.close()


# ---------------------------------------------------------------- SURVEY 8d "parity protocol at scale"
def test_config3_first_2000_proposals_of_every_walker_T0():
    """Config 3, all 64 walkers from reset: the first 2000 proposals of every walker against BRUTE FORCE (T0: every
    ratio a quotient of LU determinants of matrices built from scratch), decision for decision."""
    from concurrent.futures import ThreadPoolExecutor
    import os
    cfg = get_config(2)
    table = table_for(cfg)
    nw, nprop = cfg["n_walkers"], 2000
    seeds = walker_seeds(nw)
    W = _pkg().Walkers.from_config(cfg, table, n_walkers=nw, log_capacity=6000)
    W.reset(seeds)

    def one(seed):
        o = OracleWalker.from_config(cfg, table, int(seed), T0)
        o.reset(cfg["init_k"])
        o.propose(nprop)
        return o.log()

    with ThreadPoolExecutor(max_workers=os.cpu_count() or 1) as ex:
        fut = [ex.submit(one, s) for s in seeds]
        W.sweep(13)                                   # >= 2000 proposals per walker (sweeps of 159 ... 250)
        olog = [f.result() for f in fut]
    for w in range(nw):
        dl = W.get_log(w)
        assert len(dl) >= nprop
        compare_logs(dl[:nprop], olog[w], f"config 3 walker {w} vs T0")


def _log_replay(cfg_index, golden_seeds, n_sweeps, delay, window, n_windows):
    """Device chain from the oracle-thermalised start, `n_sweeps` sweeps in the launch configuration bench.py times;
    windows of consecutive proposals of the DEVICE log (first sweep, middle, last) re-derived by brute-force
    determinants (parity_helpers.brute_force_verify), then P7 on the final N."""
    from parity_helpers import brute_force_verify
    cfg = get_config(cfg_index)
    table = table_for(cfg)
    pkg = _pkg()
    states = [load_thermalised(cfg["name"], sd) for sd in golden_seeds]
    nw = len(states)
    seeds = walker_seeds(nw, first=50)
    W = pkg.Walkers(cfg["Lx"], cfg["Ly"], cfg["beta"], cfg["U"], cfg["K"], table, delay=delay, n_walkers=nw, init_k=0,
                    max_k=cfg["max_k"], rebuild_every=cfg["rebuild_every"], log_capacity=(n_sweeps + 1) * cfg["max_k"])
    W.set_state(seeds, [s[0] for s in states], [s[1] for s in states], [s[2] for s in states])
    W.sweep(n_sweeps)
    for w in range(nw):
        log = W.get_log(w)
        n = len(log)
        assert n > n_windows * window and W.get_stats(w)["sweeps"] == n_sweeps
        starts = [int(round(i * (n - window) / (n_windows - 1))) for i in range(n_windows)]
        worst = brute_force_verify(cfg, table, states[w][0], log, [(a, a + window) for a in starts], rtol=1e-6, atol=1e-8,
                                   what=f"{cfg['name']} delay {delay} walker {w}")
        assert worst < 1.0
        # P7: A rebuilt by the oracle from the device's final configuration; device N is its inverse
        c = W.get_config(w)
        probe = OracleWalker.from_config(cfg, table, 0, T0)
        for s in range(2):
            A = probe.A_of(s, c["site"], c["tau"], c["spin"])
            dcol = np.abs(A).max(axis=0)
            res = (A / dcol) @ (dcol[:, None] * W.get_N(w, s)) - np.eye(len(c["site"]))
            assert np.linalg.norm(res) / np.sqrt(len(c["site"])) < 1e-10
    return W


@pytest.mark.slow
def test_config4_log_replay_brute_force_windows():
    """Config 4 at full size (k ~ 1750, delay 64), 2 walkers x 30 sweeps from the thermalised start: three windows of 64
    consecutive device-log proposals per walker checked by brute-force determinants."""
    W = _log_replay(3, [0, 0], 30, 64, 64, 3)
    assert all(W.get_stats(w)["flushes"] > 300 for w in range(2))


@pytest.mark.slow
@pytest.mark.parametrize("delay", [128, 256])
def test_config5_log_replay_brute_force_windows(delay):
    """Config 5 at full size from the thermalised starts of two oracle seeds (30 sweeps each, k ~ 3600), delay 128 and
    256 (the 2-CTA cluster forms of S3), 3 sweeps: three windows of 24 consecutive device-log proposals per walker by
    brute-force determinants, P7 on the final N."""
    import os
    gdir = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    have = [sd for sd in (0, 1) if os.path.exists(os.path.join(gdir, f"thermalised_cfg5_6x6_b40_seed{sd}.txt"))]
    assert have, "tests/golden/thermalised_cfg5_6x6_b40_seed*.txt missing"
    _log_replay(4, (have * 2)[:2], 3, delay, 24, 3)
