"""gs_depth_sort_noalloc (include/gs.h): the depth sort of the binning stage as an entry point that allocates nothing --
its scratch is a static __device__ array of the library (4.2 MB, at most GS_NOALLOC_MAX_KEYS = 262 144 keys).

Checked against the EXISTING path: the depth order gs_render produces (gs_intermediates.depth_sorted: the visible Gaussians
by (depth bits, id)).  Integer work: the tolerance of the other parity tests for integers is bit-exact, and so it is here.
Two calls in a row on the shared scratch (different poses, different key counts: the second call finds the first one's
counters, histograms and status words and must clear what it needs), then the limit and the ragged sizes.

Named test_zz_*: pytest collects it last, so that with `pytest -x` a failure here hides no other test.
"""
import numpy as np
import pytest

from paper_2606_16566_b200 import binding, scenes

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def _existing_path(sc, pose):
    """gs_render through the Renderer: the unsorted keys (depth bits << 32 | id of the visible Gaussians, in id order --
    what the preprocess kernel hands to the depth sort) and the depth order the existing sort made of them."""
    from paper_2606_16566_b200.renderer import Renderer
    cam = sc.cameras[pose]
    r = Renderer(sc.P, cam.W, cam.H, 2 << 20, device="cuda:0", count_contrib=False)
    r.upload(sc)
    r.render(cam)
    torch.cuda.synchronize()
    it = r.intermediates(copy=("per_gaussian", "depth_sorted"))
    vis = np.flatnonzero(it.tiles_touched > 0)
    assert len(vis) == it.n_visible and 0 < it.n_visible <= binding.GS_NOALLOC_MAX_KEYS
    keys = (it.depth_bits[vis].astype(np.uint64) << np.uint64(32)) | vis.astype(np.uint64)
    r.close()
    return keys, it.depth_sorted.copy()


def _dev(keys_u64):
    return torch.from_numpy(keys_u64.view(np.int64).copy()).to("cuda:0")


def test_two_calls_in_a_row_match_the_depth_order_of_gs_render():
    sc = scenes.make_scene(2)                                    # 100 000 Gaussians, 800x800
    cases = [_existing_path(sc, 0), _existing_path(sc, 3)]
    assert len(cases[0][0]) != len(cases[1][0])                  # different key counts: the scratch is re-used, not re-made
    ins = [_dev(k) for k, _ in cases]
    outs = [torch.empty_like(t) for t in ins]
    torch.cuda.synchronize()
    free_before = None
    for k in range(2):                                           # back to back on one stream, no synchronisation in between
        if k == 1:
            free_before = torch.cuda.mem_get_info(0)[0]
        binding.gs_depth_sort_noalloc(ins[k], outs[k])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info(0)[0] == free_before          # the second call (module long loaded) took no device memory
    for k in range(2):
        got = outs[k].cpu().numpy().view(np.uint64)
        want = cases[k][1]
        assert got.shape == want.shape and np.array_equal(got, want), "call %d differs from gs_render's depth order" % k
        assert np.array_equal(ins[k].cpu().numpy().view(np.uint64), cases[k][0])   # the input is only read
    # and once more on the first input: the scratch now holds the second call's state
    out = torch.empty_like(ins[0])
    binding.gs_depth_sort_noalloc(ins[0], out)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy().view(np.uint64), cases[0][1])


def test_limit_ragged_sizes_and_stability():
    nmax = binding.gs_noalloc_max_keys()
    assert nmax == binding.GS_NOALLOC_MAX_KEYS == 262144
    rng = np.random.default_rng(7)
    big = torch.zeros(nmax + 1, dtype=torch.int64, device="cuda:0")
    out = torch.full((nmax + 1,), -1, dtype=torch.int64, device="cuda:0")
    with pytest.raises(binding.GsError) as ei:                   # one key too many: refused, nothing enqueued
        binding.gs_depth_sort_noalloc(big, out, nmax + 1)
    assert ei.value.code == binding.GS_ERR_LIMIT and "GS_NOALLOC_MAX_KEYS" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((out == -1).all())
    binding.gs_depth_sort_noalloc(big, out, 0)                   # nothing to do
    torch.cuda.synchronize()
    assert bool((out == -1).all())
    with pytest.raises(binding.GsError) as ei:                   # in place is not supported
        binding.gs_depth_sort_noalloc(big, big, 16)
    assert ei.value.code == binding.GS_ERR_BAD_ARG
    for n in (1, 2, 1023, 1024, 1025, 70_001, nmax):             # tile edges (1 024 keys), several tiles + a tail, the maximum
        # few distinct high words (many ties: stability is visible in the low words) mixed with full-range ones
        hi = np.where(rng.random(n) < 0.5, rng.integers(0, 50, n), rng.integers(0, 1 << 32, n)).astype(np.uint64)
        lo = rng.integers(0, 1 << 32, n).astype(np.uint64)
        keys = (hi << np.uint64(32)) | lo
        order = np.argsort(hi, kind="stable")
        t_in, t_out = _dev(keys), torch.empty(n, dtype=torch.int64, device="cuda:0")
        binding.gs_depth_sort_noalloc(t_in, t_out)
        torch.cuda.synchronize()
        assert np.array_equal(t_out.cpu().numpy().view(np.uint64), keys[order]), n


def test_the_call_can_be_captured_into_a_cuda_graph_and_replayed():
    """The use the entry point is for: under stream capture cudaMalloc is not allowed.  One warm-up call outside the capture
    (the first call on a device looks up the scratch address), then the call is captured and the graph replayed on new keys."""
    rng = np.random.default_rng(11)
    n = 50_000
    t_in = torch.zeros(n, dtype=torch.int64, device="cuda:0")
    t_out = torch.zeros(n, dtype=torch.int64, device="cuda:0")
    binding.gs_depth_sort_noalloc(t_in, t_out)
    torch.cuda.synchronize()
    side = torch.cuda.Stream(device="cuda:0")
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        graph.capture_begin()
        binding.gs_depth_sort_noalloc(t_in, t_out, stream=side)
        graph.capture_end()
    torch.cuda.synchronize()
    for rep in range(3):
        keys = rng.integers(0, 1 << 62, n, dtype=np.int64).view(np.uint64)
        t_in.copy_(_dev(keys))
        graph.replay()
        torch.cuda.synchronize()
        hi = keys >> np.uint64(32)
        assert np.array_equal(t_out.cpu().numpy().view(np.uint64), keys[np.argsort(hi, kind="stable")]), rep
