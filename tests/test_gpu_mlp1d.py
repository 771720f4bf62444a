"""The per-face MLP neural flux of one-dimensional problems (Fig. 1b; Eq. 11) and its training gradient
(Eq. 14-16): mlp1d_kernel.cuh through the C ABI.  -m gpu.

* forward: RHS and steps against the oracle's exact (fp64) MLP mode on the planar problem of 8 identical rows (the
  y-face corrections of identical rows cancel in the divergence): <= 1e-12 / <= 1e-9;
* reverse: phi = <c, S^n(U0; theta)> has gradient (J^T c, dphi/dtheta).  Exact parity against the oracle's tangent
  (O12 runs the exact MLP on the dual scalar, with a direction in its parameters): the state's adjoint and gamma_bar
  element by element against O13, the weights' gradient at sampled entries, <= 1e-11; and, independently of the
  oracle's derivative code, against central differences of its primal run (1e-5).
"""
import numpy as np
import pytest

from oracle import jxo
from paper_2601_04400_b200 import workloads as wl
from test_gpu_parity import dev, jxs, rel_err
from test_gpu_tangent import PER, smooth1d

pytestmark = pytest.mark.gpu

W = wl.mlp_weights(7)
SC = wl.mlp_scales(out_factor=5e-2)   # corrections of a few per cent of the flux: the network matters


def oracle_rows(case, w=W):
    c = wl.as_rows(case)
    o = jxo.Oracle(c["nx"], c["ny"], c["dx"], c["dy"], c["gamma"], c["mu"], c["Pr"], c["bc"])
    o.set_flux_mlp(w, *SC, emulate_bf16=False)
    return c, o


def gpu(case, w=W):
    s = jxs().Solver.from_case(case)
    s.set_flux_mlp(w, *SC)
    return s


@pytest.mark.parametrize("nx,bc", [(100, None), (255, dict(PER)), (381, dict(PER, xlo="reflective", xhi="transmissive"))])
def test_mlp1d_forward_matches_the_exact_oracle_mlp(nx, bc):
    case = wl.sod1d(nx) if bc is None else smooth1d(nx, 1e-4, bc)
    c2, o = oracle_rows(case)
    s = gpu(case)
    got = s.rhs(dev(case["U0"])).cpu().numpy()
    want = o.rhs(c2["U0"])[:, :1]
    assert rel_err(got, want) <= 1e-12
    plain = jxs().Solver.from_case(case).rhs(dev(case["U0"])).cpu().numpy()
    assert rel_err(got, plain) > 1e-4                      # the network does change the result
    U = dev(case["U0"])
    s.step(U, 0.3, 25)
    assert rel_err(U.cpu().numpy(), o.step(c2["U0"], 0.3, 25)[:, :1]) <= 1e-9
    s.set_flux_mlp(None)
    assert np.array_equal(s.rhs(dev(case["U0"])).cpu().numpy(), plain)


def test_mlp1d_training_gradient_against_differences_of_the_oracle():
    nx, ns = 96, 2
    case = smooth1d(nx, 0.0, dict(PER, xlo="transmissive", xhi="transmissive"))
    dt = 0.2 * case["dx"]
    rng = np.random.default_rng(4)
    c = rng.normal(size=case["U0"].shape)
    s = gpu(case)
    U, B = dev(case["U0"]), dev(c)
    s.step_fixed_dt_record(U, dt, ns)
    c2, o = oracle_rows(case)
    assert rel_err(U.cpu().numpy(), o.step_fixed_dt(c2["U0"], dt, ns)[:, :1]) <= 1e-12
    gbar = s.adjoint_steps(B)
    grad_u, grad_w = B.cpu().numpy(), s.flux_mlp_gradient()
    assert np.isfinite(grad_w).all() and np.abs(grad_w).max() > 0

    def phi(U0, w=W, gamma=None):
        cc = dict(case, U0=U0) if gamma is None else dict(case, U0=U0, gamma=gamma)
        c3, oo = oracle_rows(cc, w)
        return float(np.sum(c * oo.step_fixed_dt(c3["U0"], dt, ns)[:, :1]))

    # the weights: perturb the float32 parameter and divide by the step actually taken
    scale = np.abs(grad_w).max()
    picks = [0, 5, 24 * 31 + 7, 1536 + 3, 1600 + 64 * 10 + 20, 1600 + 64 * 63 + 63, 5696 + 40, 5760 + 64 + 9, 6016 + 2]
    picks += [int(j) for j in rng.integers(0, 6020, 8)]
    for j in picks:
        wp, wm = W.copy(), W.copy()
        h = np.float32(max(abs(W[j]), 0.05) * 2e-3)
        wp[j] += h
        wm[j] -= h
        fd = (phi(case["U0"], wp) - phi(case["U0"], wm)) / (float(wp[j]) - float(wm[j]))
        assert abs(grad_w[j] - fd) <= 1e-5 * scale + 1e-6 * abs(fd), (j, grad_w[j], fd)
    # the state, through the solver and through the network's input
    h = 1e-6
    for j in rng.choice(c.size, 10, replace=False):
        e = np.zeros(c.shape)
        e.flat[j] = 1.0
        fd = (phi(case["U0"] + h * e) - phi(case["U0"] - h * e)) / (2 * h)
        assert grad_u.flat[j] == pytest.approx(fd, rel=2e-5, abs=1e-7 * np.abs(grad_u).max())
    # gamma (the network's pressure input depends on it too)
    fd = (phi(case["U0"], gamma=1.4 + h) - phi(case["U0"], gamma=1.4 - h)) / (2 * h)
    assert gbar == pytest.approx(fd, rel=2e-5)


def test_mlp1d_adjoint_and_weights_gradient_match_the_transposed_oracle_tangent():
    """exact parity: O13 (the transpose of the oracle's tangent, which covers the exact MLP) for the state and gamma,
    and <Ubar, dS/dtheta_j> from the oracle's tangent along unit directions in the parameters, sampled"""
    nx, ns = 80, 2
    case = smooth1d(nx, 1e-4, dict(PER, xlo="reflective", xhi="transmissive"))
    dt = 0.2 * case["dx"]
    rng = np.random.default_rng(6)
    Ubar = rng.normal(size=case["U0"].shape)
    c2, o = oracle_rows(case)
    want, gwant = o.step_fixed_dt_adjoint(c2["U0"], Ubar, dt, ns, planar=True)
    s = gpu(case)
    U, B = dev(case["U0"]), dev(Ubar)
    s.step_fixed_dt_record(U, dt, ns)
    gbar = s.adjoint_steps(B)
    assert rel_err(B.cpu().numpy(), want) <= 1e-11
    assert gbar == pytest.approx(gwant, rel=1e-10)
    grad = s.flux_mlp_gradient()
    scale = np.abs(grad).max()
    picks = [3, 24 * 40 + 11, 1536 + 63, 1600 + 64 * 5 + 50, 5696 + 1, 5760 + 3 * 64 + 33, 6016] + \
            [int(j) for j in rng.integers(0, 6020, 10)]
    zero = np.zeros_like(c2["U0"])
    for j in picks:
        e = np.zeros(6020)
        e[j] = 1.0
        o.set_flux_mlp_direction(e)
        _, D = o.step_fixed_dt_tangent(c2["U0"], zero, 0.0, dt, ns)
        assert abs(grad[j] - float(np.sum(Ubar * D[:, :1]))) <= 1e-11 * scale, j
    # checkpointed recording: the same numbers to round-off (with the network the sums over faces are atomic)
    s.set_adjoint_checkpointing(True)
    U2, B2 = dev(case["U0"]), dev(Ubar)
    s.step_fixed_dt_record(U2, dt, ns)
    assert s.adjoint_steps(B2) == pytest.approx(gbar, rel=1e-12)
    assert np.array_equal(U2.cpu().numpy(), U.cpu().numpy()) and rel_err(B2.cpu().numpy(), B.cpu().numpy()) <= 1e-13
    assert np.abs(s.flux_mlp_gradient() - grad).max() <= 1e-13 * scale


@pytest.mark.parametrize("ckpt", [False, True])
def test_eq14_loss_over_the_unrolled_steps_and_its_gradients(ckpt):
    """jxs_adjoint_steps_mse: L = (1/m) sum_s mean((U^{n+s} - target_s)^2), Eq. 14 with its intermediate losses.
    Against the oracle: the value from its primal trajectory, dL/dgamma and dL/dtheta_j from its tangents at every
    step (L' = (1/m) sum_s mean(2 (U_s - target_s) Udot_s)), dL/dU^n from the transposes O13 of the s-step maps."""
    import torch
    nx, m = 48, 3
    case = smooth1d(nx, 0.0, dict(PER))
    dt = 0.2 * case["dx"]
    rng = np.random.default_rng(9)
    targets = case["U0"][None] + 0.05 * rng.normal(size=(m,) + case["U0"].shape)
    s = gpu(case)
    s.set_adjoint_checkpointing(ckpt)
    U, B = dev(case["U0"]), dev(np.zeros_like(case["U0"]))
    s.step_fixed_dt_record(U, dt, m)
    loss, gbar = s.adjoint_steps_mse(torch.tensor(targets, device="cuda"), B)
    grad = s.flux_mlp_gradient()
    c2, o = oracle_rows(case)
    # the oracle's trajectory and residuals
    res = []
    for k in range(1, m + 1):
        res.append(o.step_fixed_dt(c2["U0"], dt, k)[:, :1] - targets[k - 1])
    n = res[0].size
    assert loss == pytest.approx(sum(float(np.mean(r * r)) for r in res) / m, rel=1e-12)
    zero = np.zeros_like(c2["U0"])

    def dloss(Udot, gdot):
        return sum(float(np.sum(2.0 * r * o.step_fixed_dt_tangent(c2["U0"], Udot, gdot, dt, k + 1)[1][:, :1]))
                   for k, r in enumerate(res)) / (m * n)

    assert gbar == pytest.approx(dloss(zero, 1.0), rel=1e-10)
    scale = np.abs(grad).max()
    for j in [7, 1536 + 20, 1600 + 64 * 33 + 2, 5760 + 100, 6019]:
        e = np.zeros(6020)
        e[j] = 1.0
        o.set_flux_mlp_direction(e)
        assert abs(grad[j] - dloss(zero, 0.0)) <= 1e-11 * scale, j
    o.set_flux_mlp_direction(None)
    want = sum(o.step_fixed_dt_adjoint(c2["U0"], 2.0 * r / (m * n), dt, k + 1, planar=True)[0] for k, r in enumerate(res))
    assert rel_err(B.cpu().numpy(), want) <= 1e-11


def test_unrolled_training_of_the_neural_flux_reduces_the_loss():
    """P:L112-128 on the paper's own set-up (Fig. 3c-f), scaled down: a low-resolution Sod run (N = 125) with the
    neural flux is trained, m = 10 unrolled steps, towards the block-averaged high-resolution run (N = 250, Eq. 14);
    every forward and backward step runs in the kernels, the update of the weights is plain gradient descent here."""
    import torch
    nlo, m = 125, 10
    dt = 0.2 / nlo
    hi = wl.sod1d(2 * nlo)
    Uh = dev(hi["U0"])
    fine = jxs().Solver.from_case(hi)
    fine.step_fixed_dt(Uh, 0.5 * dt, 40)                                   # a developed high-resolution state ...
    start = 0.5 * (Uh[:, :, 0::2] + Uh[:, :, 1::2]).contiguous()          # ... block-averaged: the low-resolution start
    targets = torch.empty((m, 4, 1, nlo), dtype=torch.float64, device="cuda")
    for k in range(m):                                                     # d(U_HR^{n+s}), s = 1 .. m (Eq. 14)
        fine.step_fixed_dt(Uh, 0.5 * dt, 2)
        targets[k] = 0.5 * (Uh[:, :, 0::2] + Uh[:, :, 1::2])
    target = targets[-1]
    case = wl.sod1d(nlo)
    w = (0.2 * wl.mlp_weights(11)).astype(np.float32)
    s = jxs().Solver.from_case(case)
    losses = []
    lr = None
    B = torch.empty_like(start)
    for it in range(12):
        s.set_flux_mlp(w, *SC)
        U = start.clone()
        s.step_fixed_dt_record(U, dt, m)
        loss, _ = s.adjoint_steps_mse(targets, B)                          # Eq. 14 with its intermediate losses
        losses.append(loss)
        g = s.flux_mlp_gradient()
        if lr is None:
            lr = 0.1 * np.abs(w).max() / np.abs(g).max()                 # first step: 10 % of the weights' scale
        w = (w - lr * g).astype(np.float32)
    assert all(b < a for a, b in zip(losses, losses[1:])), losses
    assert losses[-1] < 0.95 * losses[0], losses
    # and the baseline without the network, for the record: training must not end above it
    s.set_flux_mlp(None)
    U = start.clone()
    s.step_fixed_dt_record(U, dt, m)
    base, _ = s.adjoint_steps_mse(targets, B)
    assert losses[-1] <= base * 1.5


def test_mlp1d_rejects_what_it_does_not_do():
    case = wl.sod1d(64)
    s = gpu(case)
    with pytest.raises(jxs().JxsError):
        s.step_fixed_dt_tangent(dev(case["U0"]), dev(case["U0"]), 1.0, 1e-3, 1)   # forward mode: no network
    s2 = jxs().Solver.from_case(case)
    with pytest.raises(jxs().JxsError):
        s2.flux_mlp_gradient()
