"""lst_index_hits_static (include/lst_static.h) against the regular path.

Why the entry point exists: some programs that embed this library are not allowed to obtain GPU
memory while they run -- an online event filter that handed the whole card to its own pool at start-up
(a later cudaMalloc fails, or at best stalls every stream of the card while it synchronises), or a
plug-in that only ever sees device pointers somebody else owns.  The regular API allocates
(lst_create, lst_bind_workspace, the first host copy of lst_get_objects), so those programs get one
call that does not: step a0, the per-sensor hit index, with its working memory in a fixed array inside
the library.  The array is shared by all calls and is never cleared between them except for its
counters, which is exactly what can go wrong -- hence TWO calls in a row here, on events of different
sizes, each compared with what the regular chain's a0 kernels produced for the same event.

Tolerance: none.  The index is integer work (offsets, caller indices) and the sorted coordinates are
copies, so everything is compared bit for bit, like the other index / set comparisons of the suite.

The file is named so that pytest collects it last: with `pytest -x` a failure here cannot hide any
other test.  It holds no state from other tests and passes alone in a fresh process as well.
"""
import numpy as np
import pytest

import lstgen

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2209_13711_b200 import binding
    binding.lib()
    return binding


def _regular_index(B, geom, mp, ev):
    """a0 of the regular chain (k_hist / k_scatter / k_rank inside lst_run) read back through the test hook."""
    lst = B.LST(geom, mp[0], mp[1], n_slots=1, max_hits=max(ev.n_hits, 1), max_seeds=1)
    lst.lst_load_event(0, ev.x, ev.y, ev.z, ev.det, None)
    lst.lst_run(0)
    out = lst.lst_test_get_hit_index(0)
    lst.close()
    return out


class _CallerBuffers:
    """Everything the caller of the allocation-free entry point has to own, made ONCE up front (this is the
    test playing the part of the host program's memory pool; the entry point itself gets addresses only)."""

    def __init__(self, torch, phic, max_hits):
        dev = "cuda:0"
        self.torch = torch
        self.n_dets = 2 * len(phic)
        self.phic = torch.from_numpy(np.ascontiguousarray(phic, np.float32)).to(dev)
        self.x, self.y, self.z = (torch.zeros(max_hits, dtype=torch.float32, device=dev) for _ in range(3))
        self.det = torch.zeros(max_hits, dtype=torch.int32, device=dev)
        self.det_off = torch.empty(self.n_dets + 1, dtype=torch.int32, device=dev)
        self.hit_orig = torch.empty(max_hits, dtype=torch.int32, device=dev)
        self.hit_xyzr = torch.empty((max_hits, 4), dtype=torch.float32, device=dev)
        self.n_rejected = torch.empty(1, dtype=torch.int32, device=dev)
        self.stage = {k: torch.empty(max_hits, dtype=torch.float32 if k != "det" else torch.int32).pin_memory()
                      for k in ("x", "y", "z", "det")}

    def upload(self, x, y, z, det):
        n = len(x)
        for k, a in (("x", x), ("y", y), ("z", z)):
            self.stage[k][:n] = self.torch.from_numpy(np.ascontiguousarray(a, np.float32))
            getattr(self, k)[:n].copy_(self.stage[k][:n])
        self.stage["det"][:n] = self.torch.from_numpy(np.ascontiguousarray(det, np.uint32).view(np.int32))
        self.det[:n].copy_(self.stage["det"][:n])
        # poison the outputs so that an entry the call fails to write cannot pass by luck
        self.det_off.fill_(-1)
        self.hit_orig.fill_(-1)
        self.hit_xyzr.fill_(float("nan"))
        self.n_rejected.fill_(-1)
        return n

    def run(self, B, n):
        B.lst_index_hits_static(self.x, self.y, self.z, self.det, self.phic, self.det_off, self.hit_orig, self.hit_xyzr,
                                self.n_rejected, n_hits=n)

    def results(self, n):
        self.torch.cuda.synchronize()
        u32 = lambda t: t.cpu().numpy().view(np.uint32)
        return u32(self.det_off), u32(self.hit_orig)[:n], self.hit_xyzr.cpu().numpy()[:n], int(self.n_rejected.item())


def test_static_scratch_index_equals_regular_path_on_two_calls_in_a_row(B, geom_full, map_full):
    import torch
    # a busy event, then a much smaller one, then the busy one again: the second call starts from the
    # first call's leftovers in every block of the shared array, the third from the second's
    big = lstgen.make_event(geom_full, "cfg3")
    small = lstgen.make_event(geom_full, "cfg3", seed=4242, n_particles=300)
    assert small.n_hits * 4 < big.n_hits <= B.LST_STATIC_MAX_HITS
    want = {id(ev): _regular_index(B, geom_full, map_full, ev) for ev in (big, small)}

    buf = _CallerBuffers(torch, geom_full.phic, big.n_hits)
    free_before = None
    for k, ev in enumerate((big, small, big)):
        n = buf.upload(ev.x, ev.y, ev.z, ev.det)
        torch.cuda.synchronize()
        if k > 0:        # the first call may load the library's device code; afterwards free memory must not move
            free_before = torch.cuda.mem_get_info()[0]
        buf.run(B, n)
        det_off, hit_orig, hit_xyzr, n_rej = buf.results(n)
        if k > 0:
            assert torch.cuda.mem_get_info()[0] >= free_before, "the call took device memory"
        w_off, w_orig, w_xyzr = want[id(ev)]
        assert n_rej == 0
        assert np.array_equal(det_off, w_off), "call %d: det_off differs" % k
        assert int(det_off[-1]) == n
        assert np.array_equal(hit_orig, w_orig), "call %d: hit_orig differs" % k
        assert np.array_equal(hit_xyzr.view(np.uint32), w_xyzr.view(np.uint32)), "call %d: sorted coordinates differ" % k
        # and the index is what it claims to be: a permutation, grouped by sensor
        assert np.array_equal(np.sort(hit_orig), np.arange(n, dtype=np.uint32))
        assert np.array_equal(np.repeat(np.arange(buf.n_dets), np.diff(det_off.astype(np.int64))), ev.det[hit_orig])


def test_static_scratch_index_leaves_out_bad_sensor_ids_and_takes_an_empty_event(B, geom_barrel):
    import torch
    ev = lstgen.make_event(geom_barrel, "cfg2")
    buf = _CallerBuffers(torch, geom_barrel.phic, ev.n_hits)
    det = ev.det.copy()
    bad = np.arange(7, ev.n_hits, 97)
    det[bad] = buf.n_dets + (bad % 3)                     # sensor ids past the detector
    n = buf.upload(ev.x, ev.y, ev.z, det)
    buf.run(B, n)
    det_off, hit_orig, hit_xyzr, n_rej = buf.results(n)
    assert n_rej == len(bad) and int(det_off[-1]) == n - len(bad)
    good = np.setdiff1d(np.arange(n), bad)
    assert np.array_equal(np.diff(det_off.astype(np.int64)), np.bincount(det[good].astype(np.int64), minlength=buf.n_dets))
    kept = hit_orig[:n - len(bad)]
    assert np.array_equal(np.sort(kept), good.astype(np.uint32))
    assert np.array_equal(np.repeat(np.arange(buf.n_dets), np.diff(det_off.astype(np.int64))), det[kept])
    assert np.array_equal(hit_xyzr[:len(kept), :3], np.stack([ev.x[kept], ev.y[kept], ev.z[kept]], 1))
    # an empty event right after a full one: every offset is zero, nothing else is written
    buf.upload(ev.x[:0], ev.y[:0], ev.z[:0], det[:0])
    buf.run(B, 0)
    det_off, hit_orig, _, n_rej = buf.results(0)
    assert n_rej == 0 and not det_off.any()
    assert (buf.hit_orig.cpu().numpy() == -1).all()


def test_static_scratch_index_refuses_sizes_beyond_the_fixed_array(B, geom_barrel):
    import torch
    buf = _CallerBuffers(torch, geom_barrel.phic, 16)
    buf.upload(np.ones(16), np.ones(16), np.zeros(16), np.zeros(16, np.uint32))
    with pytest.raises(B.LstStaticError) as e:
        buf.run(B, B.LST_STATIC_MAX_HITS + 1)
    assert e.value.status == B.LST_EINVAL and "LST_STATIC_MAX_HITS" in str(e.value) and str(B.LST_STATIC_MAX_HITS) in str(e.value)
    with pytest.raises(B.LstStaticError) as e:
        B.lst_index_hits_static(buf.x, buf.y, buf.z, buf.det, buf.phic, buf.det_off, buf.hit_orig, buf.hit_xyzr,
                                buf.n_rejected, n_hits=16, n_dets=B.LST_STATIC_MAX_DETS + 2)
    assert e.value.status == B.LST_EINVAL and "LST_STATIC_MAX_DETS" in str(e.value)
    torch.cuda.synchronize()
    assert (buf.det_off.cpu().numpy() == -1).all() and int(buf.n_rejected.item()) == -1     # nothing was enqueued
