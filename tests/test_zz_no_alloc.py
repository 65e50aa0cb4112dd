"""pespace_response_noalloc (include/pespace.h): the response entry point that allocates nothing -- its scratch is a
static device array of PESPACE_NOALLOC_SCRATCH_BYTES inside the library -- against the existing pespace_response, which
takes the same scratch from cudaMallocAsync.  Same kernels, so the outputs must agree within the response tolerance of
the parity tests (1e-8 of the channel maximum; in fact bit for bit), on two calls in a row that share the array: the
second call is smaller, has another model and other parameters, and finds the first call's constants in the scratch.

The file sorts last on purpose (pytest -x: a failure here hides nothing)."""
import ctypes as C

import numpy as np
import pytest

from paper_2602_12011_b200 import workloads as W

TOL_RESP = 1e-8          # tests/test_gpu_parity.py: relative to the channel maximum


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def test_noalloc_limits_are_checked_before_any_cuda_call():
    """sizes beyond the static array are rejected with PESPACE_ETOOBIG and a message that names them (no GPU needed:
    the check precedes every CUDA call); the stated limits of include/pespace.h are the real ones"""
    from paper_2602_12011_b200 import binding as P
    L = P.lib()
    EINVAL, ETOOBIG = -1, -4
    fake = 0x1000                                            # never dereferenced
    one = W.Model(W.MODES_22_ONLY, (W.lisa_like(),))
    three = W.Model(W.MODES_HM, (W.lisa_like(), W.taiji_like(), W.tianqin_like()))
    eight = W.Model(W.MODES_HM, tuple([W.lisa_like()] * 8))
    for model, bmax in ((one, 2016), (three, 1152), (eight, 556)):
        assert P.noalloc_scratch_needed(bmax, model) <= P.NOALLOC_SCRATCH_BYTES < P.noalloc_scratch_needed(bmax + 1, model)
        m, keep = P._model(model)
        assert L.pespace_response_noalloc(fake, bmax + 1, fake, 64, C.byref(m), fake, None) == ETOOBIG
        msg = L.pespace_strerror(ETOOBIG).decode()
        assert str(bmax + 1) in msg and str(P.NOALLOC_SCRATCH_BYTES) in msg
    m, keep = P._model(one)
    assert P.noalloc_scratch_needed(0, one) == 0
    assert L.pespace_response_noalloc(None, 4, fake, 64, C.byref(m), fake, None) == EINVAL
    assert L.pespace_response_noalloc(fake, 0, fake, 64, C.byref(m), fake, None) == EINVAL
    assert L.pespace_response_noalloc(fake, 4, fake, 0, C.byref(m), fake, None) == EINVAL
    assert L.pespace_response_noalloc(fake, 4, fake, 64, C.byref(m), None, None) == EINVAL


@pytest.mark.gpu
def test_noalloc_response_matches_the_allocating_path_on_two_calls_in_a_row():
    import torch
    from paper_2602_12011_b200 import binding as P
    import oracle
    assert torch.cuda.is_available()
    # call 1: three detectors of both kinds, five modes (response_fused_kernel), several sample tiles + ragged tails
    rng = np.random.default_rng(71)
    m1 = W.Model(W.MODES_HM, (W.lisa_like(), W.tianqin_like(), W.taiji_like(15)))
    th1 = W.draw_prior(150, 4e5, rng)
    th1[17, 4] = -1.0                                        # an out-of-domain sample: NaN row on both paths
    f1 = W.Grid(1.1e-4, 2.3e-5, 1100).freqs()
    # call 2: one detector, one mode (response_kernel), fewer samples, other parameters, other frequencies
    m2 = W.Model(W.MODES_22_ONLY, (W.lisa_like(),))
    th2 = W.draw_prior(37, 4e5, rng)
    f2 = W.Grid(1.3e-4, 3.1e-5, 700).freqs()
    f2[3] = 0.0                                              # f <= 0: zeros on both paths
    cases = [(m1, dev(th1), dev(f1)), (m2, dev(th2), dev(f2))]
    want = [torch.view_as_real(P.response(t, f, m)).clone() for m, t, f in cases]      # existing path
    outs = [torch.full_like(w, 7.0) for w in want]

    def two_calls():
        for (m, t, f), o in zip(cases, outs):
            o.fill_(7.0)
            P.response_noalloc(t, f, m, o)
        torch.cuda.synchronize()

    def compare():
        for w, o in zip(want, outs):
            w_, o_ = w.cpu().numpy(), o.cpu().numpy()
            assert np.array_equal(np.isnan(w_), np.isnan(o_))
            ok = ~np.isnan(w_)
            scale = np.abs(np.nan_to_num(w_)).max(axis=(3, 4), keepdims=True) + np.zeros_like(w_)   # per (sample, detector, channel)
            assert np.all(np.abs(o_[ok] - w_[ok]) <= TOL_RESP * scale[ok])
            assert np.array_equal(o_[ok], w_[ok])            # the same kernels on the same inputs: bit for bit

    two_calls()                                              # first use: module load, shared-memory opt-in
    compare()
    assert torch.isnan(outs[0][17]).all() and not torch.isnan(outs[0][16]).any()
    assert (outs[1][..., 3, :] == 0.0).all()
    # again, back to back, with the array holding call 2's constants when call 1 starts; the calls allocate nothing:
    # the free device memory does not move (the output buffers exist already)
    free0 = torch.cuda.mem_get_info()[0]
    n0 = P.launch_count()
    two_calls()
    assert torch.cuda.mem_get_info()[0] >= free0
    assert P.launch_count() - n0 == 4                        # prep + response kernel per call, nothing else
    compare()
    # and the oracle agrees with what came out (a few samples; the parity tests cover the kernels at large)
    got = torch.view_as_complex(outs[1]).cpu().numpy()[:3]
    ref = oracle.response(th2[:3], f2, m2)
    for b in range(3):
        for c in range(3):
            assert np.abs(got[b, 0, c] - ref[b, 0, c]).max() <= TOL_RESP * np.abs(ref[b, 0]).max()
    # a batch beyond the array is refused with a message, and nothing was written
    big = dev(W.draw_prior(2017, 4e5, rng))
    o = torch.full((2017, 1, 3, 8, 2), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(P.PespaceError, match="2017"):
        P.response_noalloc(big, dev(f2[:8]), m2, o)
    torch.cuda.synchronize()
    assert (o == 7.0).all()
