"""Host-side thread safety of libpespace.so: several host threads, each with its own CUDA stream, its own workspace and
its own batch, call the library at the same time (ctypes releases the GIL for the duration of a call).  The library
keeps no per-call global state -- the shared-memory opt-in of a kernel is an atomic per-device flag, the launch counter
is atomic, the error text is thread-local -- so every thread must get, bit for bit, what the same calls give one after
the other.  (pespace_response_noalloc is the documented exception: its calls share one scratch array and must not
overlap; it is not part of this test.)"""
import threading

import numpy as np
import pytest

from paper_2602_12011_b200 import workloads as W

pytestmark = pytest.mark.gpu

N_THREADS = 4
ROUNDS = 25


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def test_concurrent_host_threads_on_their_own_streams():
    import torch
    from paper_2602_12011_b200 import binding as P
    assert torch.cuda.is_available()
    jobs = []
    for t in range(N_THREADS):
        wl = W.config(2 + t % 3, B=40 + 9 * t, N=3000 + 257 * t)           # configs 2, 3, 4, 2: one and three detectors
        psd = wl.psd()
        data = W.coloured_noise(psd, wl.grid.df, np.random.default_rng(20 + t))
        jobs.append({"wl": wl, "theta": dev(wl.params), "data": dev(data), "psd": dev(psd),
                     "f": dev(wl.grid.freqs()[::5].copy())})
    torch.cuda.synchronize()

    def work(job, stream):
        """one thread's calls; `stream` None = the current stream (serial reference)"""
        import contextlib
        wl = job["wl"]
        ctx = torch.cuda.stream(stream) if stream is not None else contextlib.nullcontext()
        with ctx:
            lik = P.Likelihood(job["data"], job["psd"], wl.grid, wl.model, wl.B)
            lg = P.LikelihoodGrad(job["data"], job["psd"], wl.grid, wl.model, wl.B)
            fi = P.Fisher(job["data"], job["psd"], wl.grid, wl.model, 4)
            out = None
            for r in range(ROUNDS):
                th = job["theta"] if r % 2 == 0 else job["theta"].flip(0).contiguous()
                a = lik(th).clone()
                b, c = (x.clone() for x in lg(th))
                d = torch.view_as_real(P.response(th[:3], job["f"], wl.model)).clone()
                F, g = (x.clone() for x in fi(th[:4]))
                m = lik(th, mixed=True).clone()
                out = (a, b, c, d, F, g, m)
            if stream is not None:
                stream.synchronize()
        return out

    want = [work(job, None) for job in jobs]
    torch.cuda.synchronize()
    got = [None] * N_THREADS
    errors = []

    def runner(i):
        try:
            torch.cuda.set_device(0)
            got[i] = work(jobs[i], torch.cuda.Stream())
        except Exception as exc:                                 # surfaced in the main thread below
            errors.append((i, repr(exc)))

    threads = [threading.Thread(target=runner, args=(i,)) for i in range(N_THREADS)]
    for th in threads:
        th.start()
    for th in threads:
        th.join()
    torch.cuda.synchronize()
    assert not errors, errors
    for i in range(N_THREADS):
        for w, g in zip(want[i], got[i]):
            assert torch.equal(w, g), f"thread {i}: concurrent result differs from the serial one"


def test_sessions_and_repeated_calls_do_not_leak_device_memory():
    """100 session create / set_data / call / destroy cycles and 500 calls of the allocating pespace_response leave the
    free device memory where it was (sessions own a stream, device and pinned buffers; pespace_response takes its
    scratch from the stream-ordered pool)."""
    import torch
    from paper_2602_12011_b200 import binding as P
    wl = W.config(4, B=8, N=4000)
    psd = wl.psd()
    data = W.coloured_noise(psd, wl.grid.df, np.random.default_rng(1))
    th, f = dev(wl.params), dev(wl.grid.freqs())
    out = torch.empty((wl.B, 3, 3, wl.grid.N, 2), dtype=torch.float64, device="cuda")

    def cycle(n_sessions, n_calls):
        for _ in range(n_sessions):
            ses = P.Session(wl.grid, wl.model, wl.B, want_fisher=True)
            ses.set_data(data, psd)
            ses.loglike(wl.params)
            ses.loglike_grad(wl.params)
            ses.fisher(wl.params[:2])
            ses.close()
        for _ in range(n_calls):
            P.response(th, f, wl.model, out)
        torch.cuda.synchronize()

    cycle(3, 10)                                              # first use: modules, pools
    free0 = torch.cuda.mem_get_info()[0]
    cycle(100, 500)
    free1 = torch.cuda.mem_get_info()[0]
    assert free1 >= free0 - (8 << 20), (free0, free1)         # nothing accumulates (8 MiB of slack for pool granularity)
