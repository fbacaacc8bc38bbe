"""GPU parity: the CUDA path through the C-ABI against the CPU oracle, element by element."""
import numpy as np
import pytest

from paper_1811_11481_b200 import binding as B
from paper_1811_11481_b200 import synth
from tests.parity import compare, run_gpu

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("cfg,scale", [(1, 1.0), (2, 0.25), (2, 1.0), (3, 1.0), (4, 0.2)])
def test_parity_configs(row_x, cfg, scale):
    fr = synth.generate(synth.config(cfg, scale=scale))
    t, orc, exact = compare(fr, row_x)
    assert len(orc.tracks) > 50
    assert exact, "fp32 no-FMA arithmetic in identical order: track records should be bit-identical"


def test_parity_config5_reduced(row_x):
    fr = synth.generate(synth.config(5, scale=0.1))
    compare(fr, row_x)


@pytest.mark.parametrize("cfg", [4, 5])
def test_parity_full_size_bench_configuration(row_x, cfg):
    """BASELINE.json's full sizes (config 4: 6.5 M, config 5: 15.2 M clusters) in the launch configuration bench.py
    times (same capacities): every link, start hit, tracklet table, assignment and track record against the oracle."""
    fr = synth.generate(synth.config(cfg, seed=cfg))
    t = B.Tracker(row_x, n_sectors=36, max_clusters=fr.n, max_tracklets=max(1 << 16, fr.n // 8),
                  max_tracks=max(1 << 16, fr.n // 24))
    t, orc, exact = compare(fr, row_x, tracker=t)
    assert len(orc.tracks) > 50000
    assert exact


def test_grid_policy_does_not_change_results(row_x):
    fr = synth.generate(synth.config(2, scale=0.1, seed=21))
    base = run_gpu(fr, row_x)
    a0, t0 = base.assignment(), base.tracks()
    for kw in (dict(grid_bin_y=0.7, grid_bins_per_cluster=2.0), dict(grid_bin_y=9.0, grid_bins_per_cluster=0.1),
               dict(grid_bin_z_min=40.0)):
        t = run_gpu(fr, row_x, **kw)
        assert np.array_equal(t.assignment(), a0), kw
        assert t.tracks().tobytes() == t0.tobytes(), kw


def test_determinism_and_handle_reuse(row_x):
    fr = synth.generate(synth.config(2, scale=0.2, seed=7))
    fr2 = synth.generate(synth.config(3, scale=0.1, seed=8))
    t = B.Tracker(row_x, max_clusters=max(fr.n, fr2.n), max_tracklets=max(fr.n, fr2.n) // 4)
    ref = None
    for i in range(5):
        run_gpu(fr2 if i == 2 else fr, row_x, t)
        if i == 2:
            continue
        cur = (t.assignment().tobytes(), t.tracks().tobytes(), t.intermediate(B.START_HITS).tobytes())
        ref = ref or cur
        assert cur == ref
    compare(fr2, row_x, tracker=t)


def test_edge_cases(row_x):
    t = B.Tracker(row_x, max_clusters=4096, max_tracklets=1024)
    empty = synth.Frame(np.zeros(0, synth.CLUSTER_DTYPE), np.zeros(37, np.int32), np.zeros(0, np.int32),
                        np.zeros((0, 8)), 36, "empty")
    run_gpu(empty, row_x, t)
    assert t.header() == dict(n_tracks=0, n_tracklets=0, n_start_hits=0, status=0)
    # one cluster, and clusters in a single sector only
    fr = synth.generate(synth.config(2, scale=0.002, seed=3))
    compare(fr, row_x, tracker=t)
    one = synth.Frame(fr.clusters[:1].copy(), np.r_[0, np.ones(36, np.int32)].astype(np.int32), fr.truth[:1],
                      fr.track_par, 36, "one")
    compare(one, row_x, tracker=t)
    # invalid row: ignored, status bit set, assignment -1
    bad = fr.clusters.copy()
    bad["row"][5] = 999
    fb = synth.Frame(bad, fr.sector_offsets, fr.truth, fr.track_par, 36, "bad")
    run_gpu(fb, row_x, t)
    assert t.header()["status"] & 4 and t.assignment()[5] == -1
    # non-finite coordinates: ignored like a bad row (A21), the rest of the frame is tracked as if they were absent
    nf = fr.clusters.copy()
    nf["y"][7] = np.inf
    nf["z"][11] = np.nan
    nf["y"][13] = -np.inf
    run_gpu(synth.Frame(nf, fr.sector_offsets, fr.truth, fr.track_par, 36, "nonfinite"), row_x, t)
    assert t.header()["status"] & 4 and (t.assignment()[[7, 11, 13]] == -1).all()
    a_nf = t.assignment()
    keep = np.ones(fr.n, bool)
    keep[[7, 11, 13]] = False
    so2 = np.searchsorted(np.flatnonzero(keep), fr.sector_offsets).astype(np.int32)
    t2, orc2, _ = compare(synth.Frame(fr.clusters[keep], so2, fr.truth[keep], fr.track_par, 36, "without"), row_x, tracker=t)
    assert np.array_equal(a_nf[keep], orc2.assignment)
    # n > max_clusters is refused
    big = synth.generate(synth.config(2, scale=0.05, seed=3))
    with pytest.raises(B.TpccaError):
        run_gpu(big, row_x, t)


def test_boundary_argument_checks(row_x):
    """Every tpcca_get_intermediate id honours `bytes` (a short dst is refused, nothing is written), misaligned pointers
    are refused by tpcca_track and tpcca_get_intermediate (include/tpcca.h)."""
    import torch
    fr = synth.generate(synth.config(2, scale=0.05, seed=3))
    t = run_gpu(fr, row_x)
    hd = t.header()
    ns, nt = hd["n_start_hits"], hd["n_tracks"]
    assert ns > 100 and nt > 50
    need = {B.LINK_UP_RAW: fr.n * 4, B.LINK_DOWN: fr.n * 4, B.START_HITS: ns * 4, B.TRACKLET_ROW_HITS: ns * 152 * 4,
            B.TRACKLET_INTS: ns * 16, B.TRACKLET_FLOATS: ns * 32, B.TRACK_TRACKLET: nt * 4}
    st = t._stream()
    for what, nb in need.items():
        dst = torch.full((nb // 4 + 64,), 0x5A5A5A5A, dtype=torch.int32, device="cuda")
        assert t.lib.tpcca_get_intermediate(t.h, what, dst.data_ptr(), nb - 4, st) == -1, what
        assert b"too small" in t.lib.tpcca_last_error()
        torch.cuda.synchronize()
        assert bool((dst == 0x5A5A5A5A).all()), what
        assert t.lib.tpcca_get_intermediate(t.h, what, dst.data_ptr(), nb, st) == 0, what
        torch.cuda.synchronize()
        assert bool((dst[nb // 4:] == 0x5A5A5A5A).all()) and not bool((dst[:nb // 4] == 0x5A5A5A5A).all()), what
        assert t.lib.tpcca_get_intermediate(t.h, what, dst.data_ptr() + 4, nb, st) == -1  # misaligned dst
    assert t.lib.tpcca_get_intermediate(t.h, 99, dst.data_ptr(), 1 << 20, st) == -1
    dev = t.upload(fr.clusters)
    so = np.ascontiguousarray(fr.sector_offsets, np.int32)
    args = (fr.n, so.ctypes.data, st)
    assert t.lib.tpcca_track(t.h, dev.data_ptr() + 4, *args, t.out_tracks.data_ptr(), t.out_assign.data_ptr()) == -1
    assert b"misaligned" in t.lib.tpcca_last_error()
    assert t.lib.tpcca_track(t.h, dev.data_ptr(), *args, t.out_tracks.data_ptr() + 8, t.out_assign.data_ptr()) == -1
    assert t.lib.tpcca_track(t.h, dev.data_ptr(), *args, t.out_tracks.data_ptr(), t.out_assign.data_ptr() + 2) == -1
    bad = so.copy()
    bad[5] = bad[6] + 1  # not monotone
    assert t.lib.tpcca_track(t.h, dev.data_ptr(), fr.n, bad.ctypes.data, st, t.out_tracks.data_ptr(), t.out_assign.data_ptr()) == -1
    # the handle is still usable and the debug mode gives the same result
    t.set_debug(True)
    compare(fr, row_x, tracker=t)
    t.set_debug(False)


def test_capacity_overflow_is_flagged(row_x):
    fr = synth.generate(synth.config(2, scale=0.1, seed=4))
    t = B.Tracker(row_x, max_clusters=fr.n, max_tracklets=64, max_tracks=16)
    run_gpu(fr, row_x, t)
    hd = t.header()
    assert hd["status"] & 1 and 0 < hd["n_start_hits"] <= 64 and hd["n_tracks"] <= 16
    assert t.assignment().max() < 16


def test_host_api_equals_device_api(row_x):
    import torch
    fr = synth.generate(synth.config(2, scale=0.2, seed=12))
    t = run_gpu(fr, row_x)
    a0, tr0 = t.assignment(), t.tracks()
    hc = torch.from_numpy(fr.clusters.view(np.uint8).reshape(-1).copy()).pin_memory()
    ot = torch.empty(16 + 128 * t.max_tracks, dtype=torch.uint8).pin_memory()
    oa = torch.empty(fr.n, dtype=torch.int32).pin_memory()
    t.track_host(hc, fr.n, fr.sector_offsets, ot, oa)
    nt = int(ot[:16].numpy().view(B.HEADER_DTYPE)["n_tracks"][0])
    assert nt == len(tr0)
    assert np.array_equal(oa.numpy(), a0)
    assert ot[16:16 + 128 * nt].numpy().tobytes() == tr0.tobytes()


def test_permutation_invariance_gpu(row_x):
    fr = synth.generate(synth.config(2, scale=0.1, seed=30))
    fp, p = synth.permute_within_sectors(fr, seed=5)
    a = run_gpu(fr, row_x)
    b = run_gpu(fp, row_x)
    assert np.array_equal(b.assignment(), a.assignment()[p])
    assert b.tracks().tobytes() == a.tracks().tobytes()


def test_parity_non_default_parameters(row_x):
    """Every physics parameter of DESIGN.md Table A reaches the kernels: tighter cuts, shorter gap, longer seeds."""
    fr = synth.generate(synth.config(2, scale=0.15, seed=41))
    params = dict(triplet_cut=9.0, nbr_dydx=1.0, nbr_margin_z=0.5, pick_cut=9.0, reject_cut=12.0, max_gap=2,
                  min_seed_hits=5, min_tracklet_hits=14, min_track_hits=12, edge_margin=1.0, max_sinphi=0.8,
                  qual_scale=500.0, cov0=(2.0, 2.0, 0.1, 0.5, 50.0), sigma_y=0.12, sigma_z=0.13)
    t, orc, exact = compare(fr, row_x, params=params)
    assert len(orc.tracks) > 100 and exact


def test_parity_dense_noise_overflows_candidate_lists(row_x):
    """Noise far above the track density: the neighbour windows hold more candidates than the shared-memory lists
    (NB_CAP), so the nested-loop fallback of k_neighbours and multi-pass pick-up searches are exercised."""
    cfg = synth.config(1, scale=0.5, seed=43)
    cfg["noise_frac"] = 60.0
    fr = synth.generate(cfg)
    t, orc, exact = compare(fr, row_x)
    assert fr.n > 500000 and exact
    # the same frame with > 12288 bins per slice: the slice sort keeps its counters in global memory
    t2 = run_gpu(fr, row_x, grid_bins_per_cluster=4.0, grid_bin_z_min=0.05)
    assert t2.stats()["n_bins"] > 12288 * 152
    assert np.array_equal(t2.assignment(), t.assignment()) and t2.tracks().tobytes() == t.tracks().tobytes()


def test_parity_duplicate_clusters_tie_breaks(row_x):
    """Bit-identical duplicate clusters give exact ties in cost and distance: the (ord z, ord y, input index) order
    of DESIGN.md A4 decides, identically on both sides."""
    fr = synth.generate(synth.config(2, scale=0.05, seed=44))
    cl, so = [], [0]
    for s in range(36):
        c = fr.clusters[fr.sector_offsets[s]:fr.sector_offsets[s + 1]]
        cl.append(np.concatenate([c, c[::3]]))  # every third cluster twice
        so.append(so[-1] + len(cl[-1]))
    cl = np.concatenate(cl)
    f2 = synth.Frame(cl, np.asarray(so, np.int32), np.full(len(cl), -1, np.int32), fr.track_par, 36, "dup")
    compare(f2, row_x)


def test_parity_smaller_geometry(row_x):
    """n_rows = 100 and n_sectors = 8: nothing in the kernels is tied to 152 x 36."""
    fr = synth.generate(synth.config(2, scale=0.2, seed=45))
    cl, so = [], [0]
    for s in range(8):
        c = fr.clusters[fr.sector_offsets[s]:fr.sector_offsets[s + 1]]
        cl.append(c[c["row"] < 100])
        so.append(so[-1] + len(cl[-1]))
    cl = np.concatenate(cl)
    f2 = synth.Frame(cl, np.asarray(so, np.int32), np.full(len(cl), -1, np.int32), fr.track_par, 8, "small")
    t, orc, exact = compare(f2, row_x[:100])
    assert len(orc.tracks) > 20 and exact


def test_concurrent_handles_on_two_streams(row_x):
    """Two trackers driven from two host threads on two streams (frames in flight) give the results of
    the serial call: handles share no state."""
    import threading

    import torch
    frs = [synth.generate(synth.config(2, scale=0.2, seed=51)), synth.generate(synth.config(3, scale=0.2, seed=52))]
    ref = []
    for fr in frs:
        t = run_gpu(fr, row_x)
        ref.append((t.assignment(), t.tracks().tobytes()))
    out = [None, None]

    def work(i):
        torch.cuda.set_device(0)
        fr = frs[i]
        t = B.Tracker(row_x, max_clusters=fr.n, max_tracklets=max(1024, fr.n // 4))
        hc = torch.from_numpy(fr.clusters.view(np.uint8).reshape(-1).copy()).pin_memory()
        ot = torch.empty(16 + 128 * t.max_tracks, dtype=torch.uint8).pin_memory()
        oa = torch.empty(fr.n, dtype=torch.int32).pin_memory()
        with torch.cuda.stream(torch.cuda.Stream()):
            for _ in range(4):
                t.track_host(hc, fr.n, fr.sector_offsets, ot, oa)
        nt = int(ot[:16].numpy().view(B.HEADER_DTYPE)["n_tracks"][0])
        out[i] = (oa.numpy().copy(), ot[16:16 + 128 * nt].numpy().tobytes())

    ths = [threading.Thread(target=work, args=(i,)) for i in range(2)]
    for th in ths:
        th.start()
    for th in ths:
        th.join()
    for i in range(2):
        assert np.array_equal(out[i][0], ref[i][0]) and out[i][1] == ref[i][1]


@pytest.mark.parametrize("poison", [0xFF, 0x7B])
def test_poisoned_workspace(row_x, poison):
    """The caller's workspace may hold anything: every scratch array is written before it is read (frames with 36
    sectors and with one sector, capacities well above the frame, two calls per handle)."""
    for cfg, scale, ns in ((2, 0.1, 36), (1, 0.5, 1)):
        fr = synth.generate(synth.config(cfg, scale=scale, seed=61))
        t = B.Tracker(row_x, n_sectors=ns, max_clusters=2 * fr.n + 1000, max_tracklets=fr.n, max_tracks=fr.n // 2,
                      poison=poison)
        t.out_tracks.fill_(poison)
        t.out_assign.fill_(poison)
        run_gpu(fr, row_x, t)
        compare(fr, row_x, tracker=t)


def test_parity_hand_built_scenarios(row_x):
    """The hand-built inputs of the oracle's mechanics pins (gap of 5 and 6 rows, displaced hit with default and tight
    reject_cut, two crossing helices) through the CUDA path: tiny single-sector frames, every table compared."""
    from tests import scenarios
    cases = [(scenarios.gap_helix(row_x, 5), None), (scenarios.gap_helix(row_x, 6), None),
             (scenarios.displaced_hit_helix(row_x), None),
             (scenarios.displaced_hit_helix(row_x), dict(reject_cut=4.0)),
             (scenarios.crossing_helices(row_x)[0], None)]
    # round 2: selector weight (quality, then id), sector-edge stops of E2 / E3, E3 gap rule above the start row
    for displaced in (None, "A", "B"):
        for mirror in (False, True):
            cases.append((scenarios.equal_length_crossing(row_x, displaced, mirror)[0], None))
    for inward in (False, True):
        for margin in (3.0, 0.0, 60.0):
            cases.append((scenarios.edge_helix(row_x, inward)[0], dict(edge_margin=margin)))
    cases.append((scenarios.e3_gap_above_start(row_x), dict(reject_cut=4.0)))
    # round 3 (tests/test_oracle_pins_r3.py): z-displaced seed hit either side of its float64 distance 7.93, duplicates and
    # displaced clusters in a row only the pick-up search reaches (either side of pick_cut, per axis), an inward stop inside
    # the seed, the inclusive minimum hit counts, the quality step of the selector weight
    for rc in (8.16, 7.69):
        cases.append((scenarios.displaced_hit_helix_z(row_x), dict(reject_cut=rc)))
    for pos in (None, (0, 1), (0, 200), (70, 10)):
        cases.append((scenarios.lone_row_helix(row_x, duplicate=True, dup_positions=pos)[0], None))
    for kw in (dict(dz=0.55), dict(dz=0.66), dict(dy=0.38), dict(dy=0.50)):
        cases.append((scenarios.lone_row_helix(row_x, **kw)[0], None))
    cases.append((scenarios.edge_helix(row_x, inward=True, decoy_step=1)[0], dict(edge_margin=0.5)))
    full = scenarios.mk(*scenarios.one_helix(row_x), row_x)
    for kw in (dict(min_seed_hits=150), dict(min_tracklet_hits=152), dict(min_track_hits=152)):
        cases.append((full, kw))
    for dy in (0.035, 0.05):
        cases.append((scenarios.equal_length_crossing(row_x, "A", False, dy=dy)[0], None))
    for cl, params in cases:
        t, orc, exact = compare(scenarios.frame(cl), row_x, params=params)
        assert len(orc.tracks) >= 1 and exact


def test_parity_minimum_hit_counts_one_above(row_x):
    """One more than the frame has: no tracklet (seed / tracklet minimum) or no track (track minimum), on both sides."""
    from tests import scenarios
    full = scenarios.mk(*scenarios.one_helix(row_x), row_x)
    for kw, n_valid in ((dict(min_seed_hits=151), 0), (dict(min_tracklet_hits=153), 0), (dict(min_track_hits=153), 1)):
        t, orc, exact = compare(scenarios.frame(full), row_x, params=kw)
        assert len(orc.tracks) == 0 and t.header()["n_tracklets"] == n_valid, kw


def test_parity_unequal_neighbour_windows(row_x):
    """nbr_dydx != nbr_dzdx (tests/test_oracle_pins_r3.py: brute-force triplets with a narrow y and a wide z window)."""
    from tests import scenarios
    kw = dict(nbr_dydx=0.25, nbr_margin_y=0.2, nbr_dzdx=2.5, nbr_margin_z=1.5)
    fr = synth.generate(synth.config(1, scale=0.02, seed=13), noise_frac=0.4)
    compare(fr, row_x, params=kw)
    compare(synth.generate(synth.config(2, scale=0.1, seed=14)), row_x, params=kw)
    for k2 in (dict(nbr_dydx=0.3), dict(nbr_dzdx=0.3)):
        for dy, dz in ((0.9, 0.0), (0.0, 1.2)):
            fr = scenarios.frame(scenarios.window_triplet(row_x, dy, dz))
            import oracle
            orc = oracle.track(fr.clusters, fr.sector_offsets, row_x, params=k2)
            t = run_gpu(fr, row_x, **k2)
            assert np.array_equal(t.intermediate(B.LINK_UP_RAW), orc.link_up_raw)
            assert np.array_equal(t.intermediate(B.LINK_DOWN_RAW), orc.link_down_raw)


def test_parity_exact_cost_ties(row_x):
    """Mirror-image neighbour candidates have bit-equal triplet costs: the (ord z, ord y, input index) key order of
    DESIGN.md A4 decides, in every input order (tests/test_oracle_pins.py::test_exact_ties_follow_the_key_order)."""
    from tests import scenarios
    f = np.float32
    variants = ([(51, 0.05, +0.25), (51, 0.05, -0.25), (49, 0.0, 0.0)], [(51, +0.125, 0.1), (51, -0.125, 0.1), (49, 0.0, 0.0)],
                [(51, 0.0, 0.0), (49, 0.05, +0.25), (49, 0.05, -0.25)], [(51, 0.05, 0.25), (51, 0.05, 0.25), (49, 0.0, 0.0)])
    for pts in variants:
        pts = [(50, 0.0, 0.0)] + pts
        for order in ([0, 1, 2, 3], [3, 2, 1, 0], [2, 0, 3, 1]):
            q = [pts[i] for i in order]
            cl = scenarios.mk(np.array([a[0] for a in q]), np.array([a[1] for a in q], f), np.array([a[2] for a in q], f), row_x)
            fr = scenarios.frame(cl)
            orc = oracle_links(fr, row_x)
            t = run_gpu(fr, row_x)
            assert np.array_equal(t.intermediate(B.LINK_UP_RAW), orc.link_up_raw)
            assert np.array_equal(t.intermediate(B.LINK_DOWN_RAW), orc.link_down_raw)
            assert (orc.link_up_raw >= 0).sum() == 1


def oracle_links(fr, row_x):
    import oracle
    return oracle.track(fr.clusters, fr.sector_offsets, row_x)


def test_pipelined_host_call(row_x):
    """tpcca_track_host_async / tpcca_wait (two events concurrently on one GPU): two frames in flight on ONE
    handle and one workspace give, frame by frame, the results of the device-resident call; a third submission without
    a wait and a wait without a frame are refused."""
    import torch
    frs = [synth.generate(synth.config(2, scale=0.2, seed=71)), synth.generate(synth.config(3, scale=0.2, seed=72)),
           synth.generate(synth.config(4, scale=0.05, seed=73))]
    nmax = max(f.n for f in frs)
    t = B.Tracker(row_x, max_clusters=nmax, max_tracklets=max(1024, nmax // 4))
    ref = []
    for fr in frs:
        run_gpu(fr, row_x, t)
        ref.append((t.assignment(), t.tracks().tobytes()))
    bufs = []
    for fr in frs:
        bufs.append((torch.from_numpy(fr.clusters.view(np.uint8).reshape(-1).copy()).pin_memory(),
                     torch.empty(16 + 128 * t.max_tracks, dtype=torch.uint8).pin_memory(),
                     torch.empty(fr.n, dtype=torch.int32).pin_memory()))
    assert t.lib.tpcca_wait(t.h) == -1 and b"no frame" in t.lib.tpcca_last_error()
    seq = [0, 1, 2, 0, 1, 2, 2, 0]
    done = []
    t.track_host_async(bufs[seq[0]][0], frs[seq[0]].n, frs[seq[0]].sector_offsets, bufs[seq[0]][1], bufs[seq[0]][2])
    for k in range(1, len(seq) + 1):
        if k < len(seq):
            i = seq[k]
            if seq[k] == seq[k - 1]:  # the same host buffers may not be reused while their frame is in flight
                t.wait()
                done.append(k - 1)
            t.track_host_async(bufs[i][0], frs[i].n, frs[i].sector_offsets, bufs[i][1], bufs[i][2])
            if k == 1:  # two in flight: a third is refused and changes nothing
                with pytest.raises(B.TpccaError):
                    t.track_host_async(bufs[2][0], frs[2].n, frs[2].sector_offsets, bufs[2][1], bufs[2][2])
        if (k - 1) not in done:
            t.wait()
            done.append(k - 1)
        j = seq[k - 1]
        nt = int(bufs[j][1][:16].numpy().view(B.HEADER_DTYPE)["n_tracks"][0])
        assert np.array_equal(bufs[j][2].numpy(), ref[j][0]), k
        assert bufs[j][1][16:16 + 128 * nt].numpy().tobytes() == ref[j][1], k
    # the synchronous call still works afterwards and is refused while a frame is in flight
    t.track_host_async(bufs[0][0], frs[0].n, frs[0].sector_offsets, bufs[0][1], bufs[0][2])
    with pytest.raises(B.TpccaError):
        t.track_host(bufs[1][0], frs[1].n, frs[1].sector_offsets, bufs[1][1], bufs[1][2])
    t.wait()
    t.track_host(bufs[1][0], frs[1].n, frs[1].sector_offsets, bufs[1][1], bufs[1][2])
    assert np.array_equal(bufs[1][2].numpy(), ref[1][0])


def test_calls_on_one_handle_keep_their_order_across_streams(row_x):
    """All calls on a handle share one workspace.  Frames submitted alternately on two streams, with tpcca_merge and
    tpcca_get_intermediate on a third, must still give the single-stream results: the library orders them itself
    (include/tpcca.h "Streams")."""
    import torch
    frs = [synth.generate(synth.config(2, scale=0.25, seed=81)), synth.generate(synth.config(3, scale=0.2, seed=82))]
    nmax = max(f.n for f in frs)
    t = B.Tracker(row_x, max_clusters=nmax, max_tracklets=max(1024, nmax // 4))
    ref = []
    for fr in frs:
        run_gpu(fr, row_x, t)
        t.merge()
        t.torch.cuda.synchronize()
        ref.append((t.assignment(), t.tracks().tobytes(), t.merged().tobytes(), t.intermediate(B.START_HITS)))
    bufs = [(torch.from_numpy(fr.clusters.view(np.uint8).reshape(-1).copy()).pin_memory(),
             torch.empty(16 + 128 * t.max_tracks, dtype=torch.uint8).pin_memory(),
             torch.empty(fr.n, dtype=torch.int32).pin_memory()) for fr in frs]
    streams = [torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()]
    torch.cuda.synchronize()
    for rep in range(3):
        # two frames in flight, each on its own stream, no host synchronisation in between
        for i in (0, 1):
            with torch.cuda.stream(streams[i]):
                t.track_host_async(bufs[i][0], frs[i].n, frs[i].sector_offsets, bufs[i][1], bufs[i][2])
        t.wait()
        t.wait()
        for i in (0, 1):
            nt = int(bufs[i][1][:16].numpy().view(B.HEADER_DTYPE)["n_tracks"][0])
            assert np.array_equal(bufs[i][2].numpy(), ref[i][0]), (rep, i)
            assert bufs[i][1][16:16 + 128 * nt].numpy().tobytes() == ref[i][1], (rep, i)
        # device-resident frame on one stream, merge and an intermediate on others, again without waiting in between
        i = rep % 2
        dev = t.upload(frs[i].clusters)
        sh = torch.full((len(ref[i][3]) + 4,), -1, dtype=torch.int32, device="cuda")
        torch.cuda.synchronize()
        with torch.cuda.stream(streams[0]):
            t.track(dev, frs[i].n, frs[i].sector_offsets)
        with torch.cuda.stream(streams[1]):
            t.merge()
        t._check(t.lib.tpcca_get_intermediate(t.h, B.START_HITS, sh.data_ptr(), sh.numel() * 4, streams[2].cuda_stream))
        torch.cuda.synchronize()
        assert np.array_equal(t.assignment(), ref[i][0]) and t.tracks().tobytes() == ref[i][1], rep
        assert t.merged().tobytes() == ref[i][2], rep
        assert np.array_equal(sh.cpu().numpy()[:len(ref[i][3])], ref[i][3]), rep


@pytest.mark.parametrize("world", [2, 3])
def test_sector_shards_reproduce_the_whole_frame(row_x, world):
    """one frame tracked as `world` contiguous sector ranges (one handle per range, as one rank per
    GPU would) equals the whole-frame result once the track ids are offset by the exclusive scan of the per-shard counts."""
    from paper_1811_11481_b200 import distributed as D
    fr = synth.generate(synth.config(2, scale=0.3, seed=81))
    whole = run_gpu(fr, row_x)
    a_ref, tr_ref = whole.assignment(), whole.tracks()
    parts, counts = [], []
    for r in range(world):
        cl, so, lo = D.shard_frame(fr.clusters, fr.sector_offsets, world, r)
        t = run_gpu(synth.Frame(cl.copy(), so, fr.truth[lo:lo + len(cl)], fr.track_par, 36, f"shard{r}"), row_x)
        assert t.header()["status"] == 0
        parts.append((t.assignment(), t.tracks(), lo))
        counts.append(len(parts[-1][1]))
    off = D.track_id_offsets(counts)
    a = np.full(fr.n, -1, np.int32)
    for r, (ar, trr, lo) in enumerate(parts):
        a[lo:lo + len(ar)] = D.globalise_assignment(ar, off[r])
    assert sum(counts) == len(tr_ref) and np.array_equal(a, a_ref)
    assert np.concatenate([p[1] for p in parts]).tobytes() == tr_ref.tobytes()


def _gaps_untouched(t, poison):
    """Every byte between the end of one workspace array and the start of the next (arrays start on 256-byte boundaries)
    still holds the fill pattern; returns the number of gap bytes checked."""
    import torch
    lay = t.workspace_layout()
    assert len(lay) > 40
    base_off = ((t.workspace.data_ptr() + 255) & ~255) - t.workspace.data_ptr()
    checked = 0
    for (off, nb), nxt in zip(lay, [o for o, _ in lay[1:]] + [None]):
        end = off + nb
        stop = nxt if nxt is not None else min(end + 256, t.workspace.numel() - base_off)
        assert stop >= end, (off, nb, nxt)
        if stop > end:
            gap = t.workspace[base_off + end:base_off + stop]
            assert bool((gap == poison).all()), f"workspace array at offset {off} (+{nb} bytes) was overrun"
            checked += stop - end
    return checked


@pytest.mark.parametrize("case", ["config2", "dense_noise", "tight_capacity", "loopers"])
def test_no_kernel_writes_outside_its_arrays(row_x, case):
    """Bounds check of our own (compute-sanitizer is closed on the GPU pool): the workspace is filled with a pattern, the
    whole chain track -> merge -> find_legs -> fit_legs -> estimate_time runs, and the padding behind every one of the carved arrays,
    the guard bands around the caller's output buffers and the unused tail of the outputs must be untouched."""
    import torch
    poison = 0xA5
    if case == "config2":
        fr, kw = synth.generate(synth.config(2, scale=0.25, seed=7)), {}
    elif case == "dense_noise":
        fr, kw = synth.generate(synth.config(1, scale=0.5, seed=3), noise_frac=30.0), {}
    elif case == "tight_capacity":   # capacities hit: truncation must not write past the arrays either
        fr = synth.generate(synth.config(2, scale=0.25, seed=7))
        kw = dict(max_tracklets=700, max_tracks=150)
    else:
        fr, kw = synth.generate(synth.config(3, scale=0.3, seed=3)), {}
    cap = dict(max_clusters=fr.n, max_tracklets=max(1024, fr.n // 4))
    cap.update(kw)
    t = B.Tracker(row_x, n_sectors=fr.n_sectors, poison=poison, **cap)
    G = 4096
    bufs = {}
    for name, nbytes in (("tracks", 16 + 128 * t.max_tracks), ("assign", 4 * fr.n), ("merged", 16 + 128 * t.max_tracks),
                         ("track_merged", 4 * max(1, t.max_tracks)), ("partner", 4 * max(1, t.max_tracks)),
                         ("partner_in", 4 * max(1, t.max_tracks)), ("first", max(1, t.max_tracks)), ("tags", fr.n), ("summary", 32),
                         ("leg_fits", 16 + 128 * t.max_tracks),
                         ("time_s", 16 * max(1, t.max_tracks)), ("time_m", 16 * max(1, t.max_tracks))):
        full = torch.full((nbytes + 2 * G,), poison, dtype=torch.uint8, device="cuda")
        bufs[name] = (full, full[G:G + nbytes])
    import ctypes as C
    dev = t.upload(fr.clusters)
    so = np.ascontiguousarray(fr.sector_offsets, dtype=np.int32)
    p = lambda k: bufs[k][1].data_ptr()
    for _ in range(2):
        assert t.lib.tpcca_track(t.h, dev.data_ptr(), fr.n, so.ctypes.data, t._stream(), p("tracks"), p("assign")) == 0
        mp, lp = B.default_merge_params(), B.default_leg_params()
        assert t.lib.tpcca_merge(t.h, C.byref(mp), t._stream(), p("merged"), p("track_merged")) == 0
        assert t.lib.tpcca_find_legs(t.h, C.byref(lp), t._stream(), p("partner"), p("partner_in"), p("first"), p("tags"),
                                     p("summary")) == 0
        fp = B.default_leg_fit_params()
        assert t.lib.tpcca_fit_legs(t.h, C.byref(fp), t._stream(), p("leg_fits")) == 0
        assert t.lib.tpcca_estimate_time(t.h, 2.58, 250.0, t._stream(), p("time_s"), p("time_m")) == 0
    torch.cuda.synchronize()
    hd = bufs["tracks"][1][:16].cpu().numpy().view(B.HEADER_DTYPE)[0]
    assert (hd["status"] != 0) == (case == "tight_capacity")
    assert _gaps_untouched(t, poison) > 2000
    for name, (full, view) in bufs.items():
        assert bool((full[:G] == poison).all()) and bool((full[-G:] == poison).all()), f"guard band of {name} overwritten"
    nt = int(hd["n_tracks"])
    assert nt <= t.max_tracks
    assert bool((bufs["tracks"][1][16 + 128 * nt:] == poison).all()), "track records past n_tracks were written"
    nm = int(bufs["merged"][1][:16].cpu().numpy().view(B.HEADER_DTYPE)[0]["n_tracks"])
    assert bool((bufs["merged"][1][16 + 128 * nm:] == poison).all()), "merged records past n_merged were written"
