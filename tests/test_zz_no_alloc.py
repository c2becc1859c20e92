"""tpc_merge_links_no_alloc (include/tpctrk.h): track merging (K7) for callers that cannot call cudaMalloc.  Its scratch
is a static device array of the library, shared by all calls; the entry point allocates nothing and refuses sizes
beyond TPC_NO_ALLOC_MAX_TRACKS / TPC_NO_ALLOC_MAX_BINS.  Collected last (file name): a failure here hides no other test.

The GPU test compares it with the existing path (tpc_merge_tracks / tpc_get_merged on a tracker with a workspace) on
calls in a row that share the scratch: same links, chi2 within the tolerance of the merging parity tests.
"""
import ctypes

import numpy as np
import pytest

import datagen
from paper_1712_09430_b200 import binding
from parity import run_gpu

DPHI = float(np.deg2rad(20.0))          # the angle binding.Tracker hands to tpc_tracker_create


def test_sizes_beyond_the_static_scratch_are_refused_with_their_own_error():
    """No GPU needed: the limits are checked before anything touches the device."""
    L = binding.lib()
    err = ctypes.c_int(7)
    one = ctypes.c_void_p(256)          # never dereferenced: the call is refused first
    call = lambda nsec, nrows, ntr: L.tpc_merge_links_no_alloc(nsec, nrows, DPHI, 0.5, None, one, ntr, one, one, one, one, None,
                                                               ctypes.byref(err))
    assert call(36, 159, binding.TPC_NO_ALLOC_MAX_TRACKS + 1) == binding.TPC_E_LIMIT and err.value == 0
    assert call(128, 159, 10) == binding.TPC_E_LIMIT                 # 20352 bins > TPC_NO_ALLOC_MAX_BINS
    assert 36 * 159 <= binding.TPC_NO_ALLOC_MAX_BINS
    assert call(36, 159, -1) == binding.TPC_E_ARG and call(0, 159, 1) == binding.TPC_E_ARG and call(36, 300, 1) == binding.TPC_E_ARG
    assert L.tpc_merge_links_no_alloc(36, 159, DPHI, 0.5, None, None, 5, one, one, one, one, None, None) == binding.TPC_E_ARG
    assert b"scratch" in L.tpc_strerror(binding.TPC_E_LIMIT)
    with pytest.raises(binding.TpcError, match="fixed scratch"):
        binding.merge_links_no_alloc(36, 159, DPHI, 0.5, None, 256, binding.TPC_NO_ALLOC_MAX_TRACKS + 1, 256, 256, 256, 256)


def _existing_path(ev, params=None):
    trk, tracks, ids = run_gpu(ev, params)
    trk.merge_tracks()
    return tracks, ids, trk.get_merged()


def _no_alloc(torch, ev, tracks, ids, params=None, check_free=False):
    """Inputs and outputs are the caller's (torch tensors here); poisoned outputs show what the call did not write."""
    n = int(tracks.size)
    d_tracks = torch.from_numpy(tracks.view(np.uint8).reshape(-1).copy()).cuda()
    d_ids = torch.from_numpy(np.ascontiguousarray(ids, dtype=np.uint32).view(np.int32).copy()).cuda()
    d_next = torch.full((max(n, 1),), -77, dtype=torch.int32, device="cuda")
    d_prev = torch.full((max(n, 1),), -77, dtype=torch.int32, device="cuda")
    d_chi2 = torch.full((max(n, 1),), float("nan"), dtype=torch.float32, device="cuda")
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    binding.merge_links_no_alloc(ev.n_sectors, ev.n_rows, DPHI, ev.bz, params, d_tracks, n, d_ids, d_next, d_prev, d_chi2,
                                 torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    if check_free:      # (not on a device's first call, which loads the kernels) a cudaMalloc of the scratch would take 1.7 MB
        assert free_before - torch.cuda.mem_get_info()[0] < (1 << 20)
    return d_next.cpu().numpy()[:n], d_prev.cpu().numpy()[:n], d_chi2.cpu().numpy()[:n]


@pytest.mark.gpu
def test_no_alloc_merging_equals_the_existing_path_on_calls_in_a_row():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device (no CPU fallback exists)")
    # a central event, then a small one (the scratch still holds the big one's keys, bins and partner words), then the
    # first again, then other merging parameters
    p2 = binding.default_params()
    p2.merge_max_row_gap, p2.merge_chi2 = 12, 20.0
    cases = [(2, 0, None), (1, 3, None), (2, 0, None), (2, 0, p2)]
    n_links = []
    for k, (cfg, seed, prm) in enumerate(cases):
        ev = datagen.config_event(cfg, seed=seed)
        tracks, ids, ref = _existing_path(ev, prm)
        assert 0 < tracks.size <= binding.TPC_NO_ALLOC_MAX_TRACKS
        nxt, prv, chi = _no_alloc(torch, ev, tracks, ids, prm, check_free=k > 0)
        assert np.array_equal(nxt, ref["next"]) and np.array_equal(prv, ref["prev"])
        assert np.allclose(chi, ref["chi2"], rtol=1e-4, atol=1e-5)         # tolerance of the merging parity tests ...
        assert np.array_equal(chi, ref["chi2"])                            # ... and in fact the same kernels: the same bits
        n_links.append(int((nxt >= 0).sum()))
    assert n_links[0] > 50 and n_links[0] == n_links[2] and n_links[3] < n_links[0]
    # no tracks: nothing launched, nothing written
    ev = datagen.config_event(1, seed=3)
    binding.merge_links_no_alloc(ev.n_sectors, ev.n_rows, DPHI, ev.bz, None, None, 0, None, None, None, None,
                                 torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
