"""smolgp_build_events_noalloc (include/smolgp.h): the event build for callers that cannot call cudaMalloc.  Its scratch
is a fixed file-scope device array shared by every call, so the checks are: same stream, bit for bit, as
smolgp_build_events on calls made in a row (the second smaller and shuffled, so that the first call's contents sit
in the array beyond and beneath it; the third repeats the first), the size limit, and that the call is legal under a
stream capture that forbids allocation.  Collected last (file name): a failure here hides no other test."""
import numpy as np
import pytest

from paper_2601_02527_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2601_02527_b200 import binding
    return binding


@pytest.fixture(scope="module")
def ctx(B):
    c = B.Context(0)
    yield c
    c.close()


class Out:
    """caller-owned outputs of one no-alloc call (allocated by the test, before the call)"""

    def __init__(self, K):
        import torch
        dev = torch.device("cuda:0")
        # filled with junk: every element must be written by the call
        self.t = torch.full((K,), -7.0, dtype=torch.float64, device=dev)
        self.dt = torch.full((K,), -7.0, dtype=torch.float64, device=dev)
        self.delta = torch.full((K,), -7.0, dtype=torch.float64, device=dev)
        self.meta = torch.full((K,), -1, dtype=torch.int32, device=dev)
        self.exposure = torch.full((K,), -1, dtype=torch.int32, device=dev)
        self.flags = torch.full((1,), -1, dtype=torch.int32, device=dev)

    def host(self):
        import torch
        torch.cuda.synchronize()
        meta = self.meta.cpu().numpy().view(np.uint32)
        return (self.t.cpu().numpy(), self.dt.cpu().numpy(), self.delta.cpu().numpy(), (meta & 1).astype(np.int32),
                ((meta >> 1) & 31).astype(np.int32), (meta >> 8) & 0xFFFF, self.exposure.cpu().numpy(), int(self.flags.cpu()[0]))


def _dev(ts, te, inst):
    import torch
    dev = torch.device("cuda:0")
    return (torch.tensor(ts, device=dev), None if te is None else torch.tensor(te, device=dev), torch.tensor(inst, device=dev))


def _existing(ctx, d_ts, d_te, d_inst, n_inst):
    ev = ctx.smolgp_build_events(d_ts, d_te, d_inst, n_inst) if d_te is not None else ctx.smolgp_build_events_instant(d_ts, d_inst, n_inst)
    r = ev.export()
    ev.free()
    return r


def _check(got, ref, ts, te, n_inst):
    t, dt, delta, kind, inst, zmask, exposure, flags = got
    rt, rkind, rinst, rexp = ref
    assert flags == 0
    # integer and index work, and times that are copies of the inputs: bit-exact (the tolerance of the a1 tests)
    assert np.array_equal(t, rt) and np.array_equal(kind, rkind) and np.array_equal(inst, rinst) and np.array_equal(exposure, rexp)
    assert dt[0] == 0.0 and np.array_equal(dt[1:], t[1:] - t[:-1])
    if te is None:
        assert np.all(delta == 1.0) and np.all(zmask == (1 << n_inst) - 1)  # instantaneous samples open nothing
        return
    assert np.array_equal(delta, (te - ts)[exposure])
    # zero-mask: instrument i is idle after the event (XOR scan of the instrument bits), or the event is its own
    bits = (1 << inst).astype(np.int64)
    open_after = np.bitwise_xor.accumulate(bits)
    assert np.array_equal(zmask, ((~open_after) & ((1 << n_inst) - 1)) | bits)


def test_noalloc_matches_build_events_on_calls_in_a_row(B, ctx):
    import torch
    B.smolgp_noalloc_setup(0)
    assert B.smolgp_noalloc_max_events() == 262144 and 6 << 20 < B.smolgp_noalloc_scratch_bytes() < 8 << 20
    rng = np.random.default_rng(3)
    w1 = W.make(3, N=60000, n_features=4)                      # 3 overlapping instruments, K = 120000: 118 tiles
    c1 = (w1["t_start"], w1["t_end"], w1["instrument"], 3)
    w2 = W.make(4, N=4097, n_features=4)                       # 4 instruments, ragged tail, exposures SHUFFLED:
    p = rng.permutation(4097)                                  # pass 0 and the eight radix passes all run
    c2 = (w2["t_start"][p], w2["t_end"][p], w2["instrument"][p], 4)
    free = []
    for ts, te, inst, n_inst in (c1, c2, c1):
        d = _dev(ts, te, inst)
        ref = _existing(ctx, *d, n_inst)
        out = Out(2 * ts.size)
        torch.cuda.synchronize()
        f0 = torch.cuda.mem_get_info()[0]
        B.smolgp_build_events_noalloc(0, torch.cuda.current_stream().cuda_stream, *d, n_inst, out.t, out.dt, out.delta, out.meta,
                                      out.exposure, out.flags)
        torch.cuda.synchronize()
        free.append(torch.cuda.mem_get_info()[0] - f0)
        _check(out.host(), ref, ts, te, n_inst)
    assert free[1] >= 0 and free[2] >= 0  # free device memory did not shrink (the first call may load the module lazily)


def test_noalloc_instant_samples_and_input_flags(B, ctx):
    import torch
    w = W.make("instant", N=30000, n_features=4)
    d = _dev(w["t_start"], None, w["instrument"])
    ref = _existing(ctx, *d, w["n_inst"])
    out = Out(30000)
    B.smolgp_build_events_noalloc(0, 0, *d, w["n_inst"], out.t, out.dt, out.delta, out.meta, out.exposure, out.flags)
    _check(out.host(), ref, w["t_start"], None, w["n_inst"])
    # invalid input is reported through the device word, in stream order
    ts = np.array([0.0, 10.0, 5.0]); te = np.array([8.0, 20.0, 9.0]); inst = np.zeros(3, np.int32)  # exposure 2 overlaps 0
    out = Out(6)
    B.smolgp_build_events_noalloc(0, 0, *_dev(ts, te, inst), 1, out.t, out.dt, out.delta, out.meta, out.exposure, out.flags)
    assert out.host()[-1] == 4
    te[1] = 10.0                                                                                     # t_end <= t_start
    B.smolgp_build_events_noalloc(0, 0, *_dev(ts, te, inst), 1, out.t, out.dt, out.delta, out.meta, out.exposure, out.flags)
    assert out.host()[-1] & 1


def test_noalloc_size_limit(B, ctx):
    import torch
    nmax = B.smolgp_noalloc_max_events() // 2
    w = W.make(3, N=nmax, n_features=4)                       # exactly the maximum: 256 tiles
    d = _dev(w["t_start"], w["t_end"], w["instrument"])
    out = Out(2 * nmax)
    B.smolgp_build_events_noalloc(0, 0, *d, 3, out.t, out.dt, out.delta, out.meta, out.exposure, out.flags)
    _check(out.host(), _existing(ctx, *d, 3), w["t_start"], w["t_end"], 3)
    dev = torch.device("cuda:0")
    big = (torch.zeros(nmax + 1, dtype=torch.float64, device=dev), torch.ones(nmax + 1, dtype=torch.float64, device=dev),
           torch.zeros(nmax + 1, dtype=torch.int32, device=dev))
    out = Out(2 * nmax + 2)
    with pytest.raises(B.SmolgpError) as e:
        B.smolgp_build_events_noalloc(0, 0, *big, 1, out.t, out.dt, out.delta, out.meta, out.exposure, out.flags)
    assert e.value.rc == -3 and "exceed the fixed scratch" in str(e.value) and "262144" in str(e.value)
    assert int(out.flags.cpu()[0]) == -1                      # rejected before anything was enqueued


def test_noalloc_is_legal_under_stream_capture(B, ctx):
    """capture mode 'global' makes cudaMalloc / cudaFree (and any synchronising call) by this thread an error: the entry
    point passes, and the replayed graph gives the stream again -- twice, on new inputs written into the same buffers"""
    import torch
    B.smolgp_noalloc_setup(0)
    N = 20000
    w = W.make(3, N=N, n_features=4)
    d = _dev(w["t_start"], w["t_end"], w["instrument"])
    out = Out(2 * N)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, capture_error_mode="global"):
        B.smolgp_build_events_noalloc(0, torch.cuda.current_stream().cuda_stream, *d, 3, out.t, out.dt, out.delta, out.meta, out.exposure,
                                      out.flags)
    g.replay()
    _check(out.host(), _existing(ctx, *d, 3), w["t_start"], w["t_end"], 3)
    ts2 = w["t_start"] + 12345.0
    te2 = w["t_end"] + 12345.0
    d[0].copy_(torch.tensor(ts2)); d[1].copy_(torch.tensor(te2))
    g.replay()
    _check(out.host(), _existing(ctx, *d, 3), ts2, te2, 3)
