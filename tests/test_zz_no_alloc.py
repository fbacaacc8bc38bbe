"""tpcca_clean_links_static against the existing path (collected last on purpose: `pytest -x` stops at the first failure,
and a failure here must not hide the parity tests).

The entry point exists for users who cannot give the library a workspace because they cannot allocate device memory
themselves: a component living inside a process whose framework claimed the whole GPU for its own allocator, a monitoring
task looking at another component's links, code in a real-time loop where cudaMalloc would stall the device.  Its scratch
is a fixed array inside libtpcca.so that every call on a GPU shares and that keeps the previous call's contents -- so the
test makes TWO calls in a row, on frames of different size (the larger first, so that stale counts lie beyond the second
call's tiles), and checks each against what tpcca_track produced for the same frame: cleaned links bit for bit, and the
same set of start hits (tpcca_track lists them by sector, row, z, y; the static call by ascending index).
The tensors below are allocated by the TEST, through torch: the caller owns inputs and outputs, the library allocates nothing.
"""
import numpy as np
import pytest

from paper_1811_11481_b200 import binding as B
from paper_1811_11481_b200 import build, synth


def _existing_path(fr, row_x):
    """Raw links, cleaned links and start hits of one frame from tpcca_track + tpcca_get_intermediate (input-index space)."""
    t = B.Tracker(row_x, n_sectors=fr.n_sectors, max_clusters=max(fr.n, 1024), max_tracklets=max(1024, fr.n // 4))
    t.track(t.upload(fr.clusters), fr.n, fr.sector_offsets)
    t.torch.cuda.synchronize()
    out = {k: t.intermediate(w) for k, w in (("up_raw", B.LINK_UP_RAW), ("down_raw", B.LINK_DOWN_RAW), ("up", B.LINK_UP),
                                             ("down", B.LINK_DOWN), ("starts", B.START_HITS))}
    assert t.header()["status"] == 0
    t.close()
    return out


@pytest.mark.gpu
def test_static_cleaner_matches_the_existing_path_on_two_calls_in_a_row(row_x):
    import torch
    dev = torch.device("cuda:0")
    torch.cuda.set_device(dev)
    frames = [synth.generate(synth.config(2, scale=0.25, seed=31)), synth.generate(synth.config(1, seed=32))]
    assert frames[0].n > frames[1].n > 2048 and frames[0].n % 1024 != 0  # several tiles and a ragged tail, larger frame first
    ref = [_existing_path(fr, row_x) for fr in frames]
    # caller-owned buffers, filled with a pattern no valid output contains
    bufs = []
    for fr, r in zip(frames, ref):
        n = fr.n
        bufs.append(dict(
            up_raw=torch.from_numpy(r["up_raw"]).to(dev), down_raw=torch.from_numpy(r["down_raw"]).to(dev),
            up=torch.full((n,), -7, dtype=torch.int32, device=dev), down=torch.full((n,), -7, dtype=torch.int32, device=dev),
            starts=torch.full((n,), -7, dtype=torch.int32, device=dev), n_start=torch.full((1,), -7, dtype=torch.int32, device=dev)))
    torch.cuda.synchronize()
    # two calls back to back on one stream, nothing in between: the second finds the first one's scratch contents
    for fr, b in zip(frames, bufs):
        B.clean_links_static(b["up_raw"], b["down_raw"], fr.n, b["up"], b["down"], b["starts"], b["n_start"])
    torch.cuda.synchronize()
    for k, (fr, r, b) in enumerate(zip(frames, ref, bufs)):
        assert np.array_equal(b["up"].cpu().numpy(), r["up"]), f"call {k}: cleaned up links differ"
        assert np.array_equal(b["down"].cpu().numpy(), r["down"]), f"call {k}: cleaned down links differ"
        ns = int(b["n_start"].item())
        assert ns == len(r["starts"]) > 100, (k, ns, len(r["starts"]))
        got = b["starts"].cpu().numpy()
        assert np.array_equal(got[:ns], np.sort(r["starts"])), f"call {k}: start hits differ"
        assert np.all(got[ns:] == -7), f"call {k}: wrote past the start hits it reported"
    # and once more on the first frame: same answer as before (the scratch was left in a usable state)
    b = bufs[0]
    first = (b["up"].clone(), b["down"].clone(), b["starts"].clone(), b["n_start"].clone())
    for key in ("up", "down", "starts", "n_start"):
        b[key].fill_(-7)
    B.clean_links_static(b["up_raw"], b["down_raw"], frames[0].n, b["up"], b["down"], b["starts"], b["n_start"])
    torch.cuda.synchronize()
    for a, key in zip(first, ("up", "down", "starts", "n_start")):
        assert torch.equal(a, b[key]), key


def test_static_cleaner_rejects_frames_beyond_its_fixed_scratch():
    """Size and argument checks come before any CUDA call, so this part runs without a GPU."""
    build.build()
    lib = B.load()
    import os
    import re
    hdr = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "tpcca.h")).read()
    assert int(re.search(r"#define TPCCA_STATIC_MAX_CLUSTERS (\d+)LL", hdr).group(1)) == B.STATIC_MAX_CLUSTERS
    too_many = B.STATIC_MAX_CLUSTERS + 1
    assert lib.tpcca_clean_links_static(None, None, too_many, None, None, None, None, None) == -1
    msg = lib.tpcca_last_error().decode()
    assert "TPCCA_STATIC_MAX_CLUSTERS" in msg and str(B.STATIC_MAX_CLUSTERS) in msg, msg
    assert lib.tpcca_clean_links_static(None, None, -1, None, None, None, None, None) == -1
    assert lib.tpcca_clean_links_static(None, None, 16, None, None, None, None, None) == -1  # null pointers
