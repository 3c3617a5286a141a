"""tpcca_start_hits_noalloc: the start-hit selection (S4) for callers that cannot allocate device memory.

Some users of this library run where a cudaMalloc is not an option: a processing step of an online framework
that was given its slice of GPU memory at start of run and finds nothing left to allocate (and whose
cudaMalloc / cudaFree would stall the streams of the time frames in flight), a plug-in under PyTorch's caching
allocator, a QA hook that holds a sector's two link arrays and no tpcca context.  For them the library has one
entry point whose scratch is a fixed 64 KiB array inside the library image, limited to
TPCCA_NOALLOC_MAX_CLUSTERS = 2^24 links per call.

The GPU test runs the regular path (tpcca_run, stages S1-S4, workspace and all) on seeded synthetic sectors and
then feeds ITS cleaned links to the new entry point: the start hits must be the same, element for element (this
is index work, so the bar is bit-exact like every start-hit comparison in test_gpu_parity.py; the oracle has
already been compared with the regular path there).  It makes several calls in a row without waiting in
between -- a long sector, then a short one, then an empty one, then the long one again -- because all calls
share the one scratch array and each finds the previous call's numbers in it.

This file sorts last on purpose: pytest -x stops at the first failure, and a failure here must not hide the
parity tests.  It needs no state from them: it passes alone in a fresh process and after the others.
"""
import ctypes as C

import numpy as np
import pytest

import tpcsynth

LIMIT = 1 << 24


@pytest.fixture(scope="module")
def pkg():
    import paper_2208_07412_b200 as p
    p.load_library()
    return p


def test_limit_is_enforced_before_anything_touches_the_gpu(pkg):
    """Runs on the CPU box too: a call beyond the limit (or with bad sizes) is refused by host checks alone,
    with a message that names the limit; exactly the limit passes the size check (and then fails for want of
    a device or of pointers, not for its size)."""
    from paper_2208_07412_b200 import binding
    assert binding.NOALLOC_MAX_CLUSTERS == LIMIT
    lib = pkg.load_library()
    msg = C.create_string_buffer(512)
    one = C.c_int32(0)      # stands in for n_start; never written: the call is refused first
    rc = lib.tpcca_start_hits_noalloc(0, None, None, None, LIMIT + 1, None, 0, C.byref(one), msg, len(msg))
    assert rc == -1 and str(LIMIT) in msg.value.decode() and "TPCCA_NOALLOC_MAX_CLUSTERS" in msg.value.decode()
    rc = lib.tpcca_start_hits_noalloc(0, None, None, None, -1, None, 0, C.byref(one), msg, len(msg))
    assert rc == -1 and msg.value
    rc = lib.tpcca_start_hits_noalloc(0, None, None, None, LIMIT, None, 0, C.byref(one), msg, len(msg))
    assert rc == -1 and "NULL" in msg.value.decode()          # size accepted, pointers refused
    rc = lib.tpcca_start_hits_noalloc(0, None, None, None, 0, None, 0, None, None, 0)   # no message buffer: still an error code
    assert rc == -1


@pytest.mark.gpu
def test_start_hits_match_the_regular_path_on_calls_in_a_row(pkg):
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device is visible")
    from paper_2208_07412_b200 import binding

    # the regular path: S1-S4 through tpcca_create / tpcca_run on config-1 kinematics (36 sectors, ~25 k clusters each:
    # a dozen 2048-cluster tiles and a ragged tail per sector)
    tf = tpcsynth.generate(1, n_tracks=6000)
    with pkg.Tracker(tf.params, max_clusters=tf.n_clusters) as trk:
        trk.load_timeframe(tf)
        trk.run(0x0F)
        trk.sync()
        outs = trk.get_tracks_all(binding.OUT_LINKS | binding.OUT_START)
    sizes = [o.n for o in outs]
    big, small = int(np.argmax(sizes)), int(np.argmin(sizes))
    assert sizes[big] > 5 * 2048 and sizes[big] % 2048 != 0 and sizes[small] > 0
    for o in (outs[big], outs[small]):
        assert len(o.start_hit) > 10     # there is something to compare

    dev = torch.device("cuda:0")
    # everything the calls use is created BEFORE the first call; the calls themselves allocate nothing
    cases = [big, small, None, big, small]                                    # None = an empty sector
    ins, res = [], []
    for s in cases:
        up = torch.from_numpy(outs[s].link_up if s is not None else np.zeros(0, np.int32)).to(dev)
        dn = torch.from_numpy(outs[s].link_dn if s is not None else np.zeros(0, np.int32)).to(dev)
        cap = len(outs[s].start_hit) if s is not None else 4
        ins.append((up, dn))
        res.append((torch.full((cap + 7,), -7, dtype=torch.int32, device=dev), torch.full((1,), -7, dtype=torch.int32, device=dev)))
    short = (torch.full((5,), -7, dtype=torch.int32, device=dev), torch.full((1,), -7, dtype=torch.int32, device=dev))

    binding.start_hits_noalloc(*ins[0], *res[0])          # first call on the device: includes the one-time set-up
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info(dev)[0]
    for (up, dn), (sh, ns) in zip(ins[1:], res[1:]):      # calls in a row on one stream, no waiting in between
        binding.start_hits_noalloc(up, dn, sh, ns)
    binding.start_hits_noalloc(*ins[0], *short)           # capacity smaller than the number of start hits
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info(dev)[0] == free0       # the driver's free-memory figure did not move

    for s, (sh, ns) in zip(cases, res):
        want = outs[s].start_hit if s is not None else np.zeros(0, np.int32)
        got_n = int(ns.item())
        assert got_n == len(want), (s, got_n, len(want))
        got = sh.cpu().numpy()
        assert np.array_equal(got[:got_n], want), s          # bit-exact, ascending position
        assert np.all(got[got_n:] == -7), s                  # nothing written beyond n_start
    assert int(short[1].item()) == len(outs[big].start_hit)                   # found, not stored
    assert np.array_equal(short[0].cpu().numpy(), outs[big].start_hit[:5])    # the first `capacity` hits are stored

    # a different stream than the one the inputs were made on (ordered by the synchronize above)
    st = torch.cuda.Stream(dev)
    sh, ns = torch.full_like(res[1][0], -7), torch.full_like(res[1][1], -7)
    torch.cuda.synchronize()
    binding.start_hits_noalloc(*ins[1], sh, ns, stream=st)
    st.synchronize()
    assert int(ns.item()) == len(outs[small].start_hit)
    assert np.array_equal(sh.cpu().numpy()[:int(ns.item())], outs[small].start_hit)
