"""SURVEY 8(f)-3 as a checked component: three iterations of the inverse-design harness
(paper_2603_24027_b200/optimize.py: Gaussian filter -> projection -> eps, chain rule, Nesterov-Adam) on a small coupler-shaped
problem.  Every grad_eps comes from the CUDA path (fdtd_forward + fdtd_reverse) and is compared with the oracle's gradient for
the same design; the design gradient d loss / d rho is compared with central differences of the ORACLE's float64 loss."""
import numpy as np
import pytest

from oracle import fdtd_oracle as orc
from paper_2603_24027_b200 import optimize as O, workloads as W
from tests.helpers import gpu_gradient, gpu_sim, oracle_gradient, rel_l2

pytestmark = pytest.mark.gpu


def mini_coupler(nsteps=90):
    """40x40x32 cells, 8-cell CPML: a 4-cell Si layer in SiO2, 16x16 design patch in the layer, y-polarised line source above
    it, flux monitor plane at the end of the layer — the shape of the C2 workload (BASELINE.json configs[1]) at oracle size."""
    shape, P = (40, 40, 32), 8
    eps = np.full(shape, W.EPS_SIO2, dtype=np.float32)
    eps[:, :, 14:18] = W.EPS_SI
    i = np.arange(10, 30, dtype=np.float64)
    amp = np.exp(-((i - 20.0) / 5.0) ** 2).astype(np.float32).reshape(20, 1, 1)
    src = W.Source(1, (10, 20, 21), (30, 21, 22), amp, W.gauss_sine(nsteps, 24, 8))
    return W.Workload("mini-coupler", shape, P, nsteps, eps, ((12, 12, 14), (28, 28, 18)), [src],
                      ((30, 12, 12), (31, 28, 20), 0b110110), "flux_x", W.F32, 1)


def _with_eps(w, eps):
    import dataclasses
    return dataclasses.replace(w, eps=eps)


@pytest.mark.parametrize("dtype,k", [(W.F32, 1), (W.F8E4M3B11FNUZ, 4)])
def test_three_design_iterations_gradients_match_oracle(dtype, k):
    w = mini_coupler()
    des = O.Design(w)
    rng = np.random.default_rng(5)
    rho = np.clip(0.5 + 0.2 * rng.standard_normal((des.nx, des.ny)), 0.0, 1.0)
    st = {"t": 0, "m": 0.0, "v": 0.0}
    flux = []
    for it in range(3):
        beta = 1.0 + 2.0 * it
        eps, _ = des.forward(rho, beta)
        wi = _with_eps(w, eps)
        g = gpu_gradient(wi, dtype, k, sim=gpu_sim(wi))
        o = oracle_gradient(wi, 32, dtype, k)
        err = rel_l2(g["grad"], o["grad"])
        print(f"[optimize] it {it} dtype {dtype} k {k}: loss gpu {g['L']:.6e} oracle {o['L']:.6e}, grad_eps rel-L2 {err:.3e}")
        assert np.abs(o["grad"]).max() > 0
        assert err <= 1e-4
        assert abs(g["L"] - o["L"]) <= 1e-5 * abs(o["L"])
        g_rho = des.backward(g["grad"])
        g_rho_o = des.backward(o["grad"])
        assert rel_l2(g_rho, g_rho_o) <= 1e-4
        if it == 0 and dtype == W.F32:
            # d loss / d rho against central differences of the oracle's float64 loss (native f64 store, k = 1)
            def loss64(r):
                e, _ = des.forward(r, beta)
                return oracle_gradient(_with_eps(w, e), 64, orc.NATIVE, 1)["L"]
            des.forward(rho, beta)          # restore the projection derivative of THIS rho for backward()
            g_rho = des.backward(g["grad"])
            for (a, b) in [(3, 4), (8, 8), (12, 5)]:
                h = 2e-2
                rp, rm = rho.copy(), rho.copy()
                rp[a, b] += h
                rm[a, b] -= h
                fd = (loss64(rp) - loss64(rm)) / (2 * h)
                print(f"[optimize] d loss/d rho[{a},{b}]: chain rule {g_rho[a, b]:.6e}, central difference {fd:.6e}")
                assert abs(fd - g_rho[a, b]) <= 2e-2 * max(abs(fd), np.abs(g_rho).max() * 1e-2)
            des.forward(rho, beta)
        flux.append(-g["L"])
        lr = 0.05 * min(1.0, (it + 1) / 2)
        rho = np.clip(rho - O.nadam_step(st, g_rho, lr), 0.0, 1.0)
    assert np.isfinite(flux).all()
