"""Out-of-bounds WRITE check of every entry point (compute-sanitizer is not available on the GPU pool): the caller's
workspace and output arrays are exact-size windows inside larger buffers whose margins hold a byte pattern; after the
call the margins must be untouched.  Shapes are ragged on purpose (B and N no multiples of the tile / block sizes,
fewer samples than one tile, one bin), and the workspace is exactly pespace_workspace_bytes*() long, so a kernel that
writes past the last tile, the last bin block or the last partial slice lands in a margin."""
import numpy as np
import pytest

from paper_2602_12011_b200 import workloads as W

pytestmark = pytest.mark.gpu

GUARD = 1 << 16          # bytes on either side (a multiple of 256: the window keeps the 16-byte alignment of the ABI)
PATTERN = 0xA5


@pytest.fixture(scope="module")
def P():
    import torch
    from paper_2602_12011_b200 import binding
    assert torch.cuda.is_available()
    return binding


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


class Guarded:
    """an exact-size window of `nbytes` inside a buffer with PATTERN-filled margins"""

    def __init__(self, nbytes: int):
        import torch
        self.n = int(nbytes)
        self.buf = torch.full((self.n + 2 * GUARD,), PATTERN, dtype=torch.uint8, device="cuda")
        self.win = self.buf[GUARD:GUARD + self.n]

    def f64(self, *shape):
        import torch
        assert int(np.prod(shape)) * 8 == self.n
        return self.win.view(torch.float64).view(*shape)

    def check(self, what: str):
        import torch
        torch.cuda.synchronize()
        lo, hi = self.buf[:GUARD], self.buf[GUARD + self.n:]
        assert bool((lo == PATTERN).all()), f"{what}: bytes BEFORE the array were written"
        assert bool((hi == PATTERN).all()), f"{what}: bytes AFTER the array were written"


def guard_workspace(obj) -> Guarded:
    g = Guarded(obj.ws_bytes)
    obj.ws = g.win
    return g


SHAPES = [(1, 1), (3, 257), (67, 1100), (130, 700)]          # (B, N)


def model_for(n_det: int, mask: int):
    dets = (W.lisa_like(), W.tianqin_like(), W.taiji_like(15))[:n_det]
    return W.Model(mask, dets)


def workload(B: int, N: int, n_det: int, mask: int, seed: int = 5):
    rng = np.random.default_rng(seed)
    th = W.draw_prior(B, 4e5, rng)
    return W.Workload("guard", W.Grid(1.1e-4, 2.3e-5, N), model_for(n_det, mask), th, th[0].copy(), 9)


@pytest.mark.parametrize("B,N", SHAPES)
@pytest.mark.parametrize("n_det,mask", [(1, W.MODES_22_ONLY), (1, W.MODES_HM), (3, W.MODES_HM), (2, W.MODE_33 | W.MODE_21)])
def test_loglike_response_fisher_grad_stay_inside_their_arrays(P, B, N, n_det, mask):
    wl = workload(B, N, n_det, mask)
    psd = wl.psd()
    data = W.coloured_noise(psd, wl.grid.df, np.random.default_rng(3))
    d_data, d_psd, d_th = dev(data), dev(psd), dev(wl.params)
    # pespace_loglike / pespace_loglike_mixed
    lik = P.Likelihood(d_data, d_psd, wl.grid, wl.model, B)
    gw, go = guard_workspace(lik), Guarded(8 * B)
    lik(d_th, out=go.f64(B))
    gw.check("pespace_loglike workspace"); go.check("pespace_loglike out")
    lik(d_th, out=go.f64(B), mixed=True)
    gw.check("pespace_loglike_mixed workspace"); go.check("pespace_loglike_mixed out")
    # pespace_prepare + pespace_loglike_prepared
    lik.prepare()
    gw.check("pespace_prepare workspace")
    lik(d_th, out=go.f64(B))
    assert lik.prepared
    gw.check("pespace_loglike_prepared workspace"); go.check("pespace_loglike_prepared out")
    # pespace_loglike_grad
    lg = P.LikelihoodGrad(d_data, d_psd, wl.grid, wl.model, B)
    gw, go, gg = guard_workspace(lg), Guarded(8 * B), Guarded(8 * B * 11)
    lg(d_th, out_lnL=go.f64(B), out_grad=gg.f64(B, 11))
    gw.check("pespace_loglike_grad workspace"); go.check("pespace_loglike_grad lnL"); gg.check("pespace_loglike_grad grad")
    lg.prepare()
    lg(d_th, out_lnL=go.f64(B), out_grad=gg.f64(B, 11))
    gw.check("pespace_loglike_grad_prepared workspace"); go.check("pespace_loglike_grad_prepared lnL")
    gg.check("pespace_loglike_grad_prepared grad")
    # pespace_fisher (matrix + gradient, gradient only)
    fi = P.Fisher(d_data, d_psd, wl.grid, wl.model, B)
    gw, gF, gg = guard_workspace(fi), Guarded(8 * B * 121), Guarded(8 * B * 11)
    fi(d_th, out_F=gF.f64(B, 11, 11), out_grad=gg.f64(B, 11))
    gw.check("pespace_fisher workspace"); gF.check("pespace_fisher F"); gg.check("pespace_fisher grad")
    fi(d_th, out_grad=gg.f64(B, 11), grad_only=True)
    gw.check("pespace_fisher (gradient only) workspace"); gg.check("pespace_fisher (gradient only) grad")
    # pespace_response on a frequency array of its own length
    Nf = max(1, N - 3)
    f = dev(wl.grid.freqs()[:Nf])
    gr = Guarded(16 * B * n_det * 3 * Nf)
    P.response(d_th, f, wl.model, out=gr.f64(B, n_det, 3, Nf, 2))
    gr.check("pespace_response out")


@pytest.mark.parametrize("B,N", SHAPES[1:])
@pytest.mark.parametrize("n_det,mask", [(1, W.MODES_22_ONLY), (3, W.MODES_HM), (2, W.MODE_22 | W.MODE_33 | W.MODE_44)])
def test_tabulated_paths_stay_inside_their_arrays(P, B, N, n_det, mask):
    import torch
    wl = workload(B, N, n_det, mask, seed=6)
    psd = wl.psd()
    data = W.coloured_noise(psd, wl.grid.df, np.random.default_rng(4))
    d_data, d_psd, d_th = dev(data), dev(psd), dev(wl.params)
    f = wl.grid.freqs()
    # tabulated waveforms (T1)
    table = W.chirp_table(wl.params, mask, W.log_nodes(f[0], f[-1], 97))
    d_tab = P.WaveTable(*(dev(x) for x in table))
    lt = P.LikelihoodTab(d_data, d_psd, wl.grid, wl.model, B)
    gw, go = guard_workspace(lt), Guarded(8 * B)
    lt(d_th, d_tab, out=go.f64(B))
    gw.check("pespace_loglike_tab workspace"); go.check("pespace_loglike_tab out")
    ft = P.FisherTab(d_data, d_psd, wl.grid, wl.model, B)
    gw = guard_workspace(ft)
    F, g = ft(d_th, d_tab)
    gw.check("pespace_fisher_tab workspace")
    assert F.shape == (B, 11, 11) and g.shape == (B, 11)
    Nf = max(1, N - 5)
    gr = Guarded(16 * B * n_det * 3 * Nf)
    P.response_tab(d_th, d_tab, dev(f[:Nf]), wl.model, out=gr.f64(B, n_det, 3, Nf, 2))
    gr.check("pespace_response_tab out")
    # tabulated orbits (T2)
    tab = W.synthetic_orbit_table(wl.model.detectors, -40 * 86400.0 * 30, 7200.0, 16000, seed=2)
    d_orb = P.OrbitTable(tab[0], tab[1], dev(tab[2]), dev(tab[3]))
    lo = P.LikelihoodOrb(d_data, d_psd, wl.grid, wl.model, B)
    gw, go = guard_workspace(lo), Guarded(8 * B)
    lo(d_th, d_orb, out=go.f64(B))
    gw.check("pespace_loglike_orb workspace"); go.check("pespace_loglike_orb out")
    gr = Guarded(16 * B * n_det * 3 * Nf)
    P.response_orb(d_th, d_orb, dev(f[:Nf]), wl.model, out=gr.f64(B, n_det, 3, Nf, 2))
    gr.check("pespace_response_orb out")
    torch.cuda.synchronize()
