"""The calls that allocate nothing inside -- pespace_loglike_prepared, pespace_loglike_grad_prepared (caller's workspace)
and pespace_response_noalloc (static scratch) -- captured in a CUDA graph: the launch-bound single-theta regime of a
sampler replayed without host-side launch work.  Replays must reproduce the eager calls bit for bit,
also after theta was updated in place.  Each entry point is called once before the capture (first use sets the
shared-memory opt-in of its kernels and looks the scratch address up; neither belongs inside a capture)."""
import numpy as np
import pytest

from paper_2602_12011_b200 import workloads as W

pytestmark = pytest.mark.gpu


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("idx", [2, 4])
def test_prepared_and_noalloc_calls_replay_from_a_cuda_graph(idx):
    import torch
    from paper_2602_12011_b200 import binding as P
    wl = W.config(idx, B=3, N=5000)
    psd = wl.psd()
    data = W.coloured_noise(psd, wl.grid.df, np.random.default_rng(8))
    d_data, d_psd = dev(data), dev(psd)
    th = dev(wl.params)
    f = dev(wl.grid.freqs()[:777])
    nd = len(wl.model.detectors)
    lik = P.Likelihood(d_data, d_psd, wl.grid, wl.model, wl.B).prepare()
    lg = P.LikelihoodGrad(d_data, d_psd, wl.grid, wl.model, wl.B).prepare()
    lnL = torch.empty(wl.B, dtype=torch.float64, device="cuda")
    gl, gg = torch.empty_like(lnL), torch.empty((wl.B, 11), dtype=torch.float64, device="cuda")
    resp = torch.empty((wl.B, nd, 3, 777, 2), dtype=torch.float64, device="cuda")

    def calls():
        lik(th, lnL)
        lg(th, gl, gg)
        P.response_noalloc(th, f, wl.model, resp)

    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):                            # warm-up outside the capture
        calls()
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    want = [x.clone() for x in (lnL, gl, gg, resp)]
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        calls()                                              # recorded, not run
    for x in (lnL, gl, gg, resp):
        x.fill_(-1.0)
    graph.replay()
    torch.cuda.synchronize()
    for got, w in zip((lnL, gl, gg, resp), want):
        assert torch.equal(got, w)
    # a sampler's step: new theta written into the same buffer, same graph
    new = wl.params.copy()
    new[:, 10] += 5.0
    new[:, 7] += 0.01
    th.copy_(dev(new))
    graph.replay()
    torch.cuda.synchronize()
    got = [x.clone() for x in (lnL, gl, gg, resp)]
    calls()                                                  # eager, same inputs
    torch.cuda.synchronize()
    for g_, e in zip(got, (lnL, gl, gg, resp)):
        assert torch.equal(g_, e)
    assert not torch.equal(got[0], want[0])                  # and theta did change the result
