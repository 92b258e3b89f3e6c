"""Pins for the oracle's complex path (O5: Eq. 14 contour deformation, its Jacobian, log branches).

The Jacobian of Eq. 14 is not printed in the paper.  It is pinned here WITHOUT retyping it:
torch autograd differentiates z(t) = t - i lambda t(1-t) dF/dt, and a tensor Gauss-Legendre quadrature
(no lattice, no periodisation, another lambda) integrates the deformed integrand of config 3 built from
the F polynomial as stated in SURVEY 8(d).  CPU only.
"""
import numpy as np
import pytest
import torch

import qmc_inputs as qi
from oracle import Oracle

torch.set_default_dtype(torch.float64)


def poly_fn(coeff, expo):
    def f(t):  # t: [n] real or complex; integer powers by repeated multiplication (exact derivatives at t = 0)
        tot = 0.0
        for c, e in zip(coeff, expo):
            m = torch.ones((), dtype=t.dtype) * float(c)
            for j, ej in enumerate(e):
                for _ in range(int(ej)):
                    m = m * t[j]
            tot = tot + m
        return tot
    return f


def autograd_deformation(F, lam, t):
    """z(t) and det(dz/dt) by automatic differentiation of Eq. 14."""
    t = torch.tensor(t)

    def d(tt):  # imaginary displacement, real
        g = torch.autograd.functional.jacobian(F, tt, create_graph=True)
        return -lam * tt * (1 - tt) * g
    disp = d(t)
    Jd = torch.autograd.functional.jacobian(d, t)
    z = t + 1j * disp
    det = torch.linalg.det(torch.eye(len(t), dtype=torch.complex128) + 1j * Jd)
    return z.detach().numpy(), complex(det.detach())


@pytest.mark.parametrize("wl", [qi.massive_box(), qi.nonplanar_vertex()], ids=lambda w: w.name)
def test_jacobian_determinant_matches_autograd(wl):
    o = Oracle.from_workload(wl)
    rng = np.random.default_rng(42)
    for s in range(0, o.n_sectors, max(1, o.n_sectors // 6)):
        sec = o.sector(s)
        F = poly_fn(*sec["F"])
        for _ in range(3):
            t = rng.uniform(0.02, 0.98, size=o.dim)
            z, det = o.deform(s, t)
            z2, det2 = autograd_deformation(F, wl.lam, t)
            assert np.allclose(z, z2, rtol=1e-13, atol=1e-15)
            assert abs(det - det2) <= 1e-12 * max(1.0, abs(det2))
        # corner point: components set to 0 -> z_j = 0 and the row reduces to rho_j on the diagonal
        t = rng.uniform(0.1, 0.9, size=o.dim)
        t[0] = 0.0
        z, det = o.deform(s, t)
        z2, det2 = autograd_deformation(F, wl.lam, t)
        assert z[0] == 0 and abs(det - det2) <= 1e-12 * max(1.0, abs(det2))


def cfg3_sector_polys():
    """Primary sectors of F = -5x2x4 + 1.5x1x3 - 0.52x2x3 - 0.52x3x4 + (x1+x2+x3+x4)^2."""
    def F(x):
        return (-5 * x[1] * x[3] + 1.5 * x[0] * x[2] - 0.52 * x[1] * x[2] - 0.52 * x[2] * x[3]
                + (x[0] + x[1] + x[2] + x[3]) ** 2)
    out = []
    for l in range(4):
        def Fl(t, l=l):  # t: [..., 3]
            xs = list(torch.unbind(t, dim=-1))
            xs.insert(l, torch.ones_like(xs[0]))
            return F(xs)
        out.append(Fl)
    return out


def gl_nodes(n, dim):
    x, w = np.polynomial.legendre.leggauss(n)
    x = 0.5 * (x + 1); w = 0.5 * w
    grids = np.meshgrid(*([x] * dim), indexing="ij")
    pts = np.stack([g.ravel() for g in grids], axis=1)
    wts = np.prod(np.stack(np.meshgrid(*([w] * dim), indexing="ij")), axis=0).ravel()
    return pts, wts


def torch_gl_J0(lam, nodes=32):
    """J_0 = sum_l int d^3t det(dz/dt) F_l(z)^-2 (a_U0 = 0, a_F0 = -2) by tensor Gauss-Legendre + autograd."""
    pts, wts = gl_nodes(nodes, 3)
    t = torch.tensor(pts, requires_grad=True)
    w = torch.tensor(wts)
    total = 0j
    for Fl in cfg3_sector_polys():
        val = Fl(t)
        (g,) = torch.autograd.grad(val.sum(), t, create_graph=True)
        disp = -lam * t * (1 - t) * g                       # [M,3] real
        rows = []
        for i in range(3):
            (r,) = torch.autograd.grad(disp[:, i].sum(), t, retain_graph=True)
            rows.append(r)
        Jd = torch.stack(rows, dim=1)                       # [M,3,3], d disp_i / d t_k
        J = torch.eye(3, dtype=torch.complex128) + 1j * Jd.detach()
        z = (t + 1j * disp).detach()
        Fz = Fl(z)
        assert float(Fz.imag.max()) <= 0.0                  # contour on the right side
        total += complex((w * torch.linalg.det(J) / Fz ** 2).sum())
    return total


SURVEY_CFG3 = 0.29347155740583 + 0.33214829595148j   # SURVEY 8(c) "O5 deformation" (iv)


def test_config3_gauss_legendre_pin():
    ref = torch_gl_J0(0.3)
    assert abs(ref - torch_gl_J0(0.7, nodes=36)) < 2e-11      # lambda-independence of the pin itself
    assert abs(ref - SURVEY_CFG3) < 2e-11
    # (a) the oracle's deformed integrand (lambda = 0.5) summed with the same Gauss-Legendre rule
    o = Oracle.from_workload(qi.massive_box())
    pts, wts = gl_nodes(32, 3)
    tot = 0j
    for s in range(4):
        tot += sum(wt * o.sector_integrand(s, p)[0] for p, wt in zip(pts, wts))
    assert abs(tot - ref) < 2e-11
    # (b) the oracle's lattice estimate within 3 sigma
    N = 32749
    S, A, cnt = o.integrate(N, qi.good_vector(N, 3), qi.splitmix64_shifts(11, 8, 3))
    coeff, err = o.totals(S)
    assert cnt[0] == 0 and cnt[1] == 0 and cnt[2] == 0       # F quadratic in t: Im F(z) <= 0 exactly
    assert abs(coeff[0].real - ref.real) <= 3 * err[0].real and abs(coeff[0].imag - ref.imag) <= 3 * err[0].imag
    assert err[0].real < 2e-6 and err[0].imag < 2e-6


def test_below_threshold_imaginary_part_vanishes():
    # s = 3 < 4 m^2: F > 0 on the whole cube, so the deformed result equals the undeformed real one
    pts, wts = gl_nodes(24, 3)
    wl = qi.massive_box(s=3.0)
    oc = Oracle.from_workload(wl, lam=0.5)
    orr = Oracle.from_workload(wl, lam=0.0)
    c = sum(wt * oc.sector_integrand(s, p)[0] for s in range(4) for p, wt in zip(pts, wts))
    r = sum(wt * orr.sector_integrand(s, p)[0] for s in range(4) for p, wt in zip(pts, wts))
    assert r.imag == 0.0
    assert abs(c.imag) < 1e-10 and abs(c.real - r.real) < 1e-10
    assert r.real == pytest.approx(0.268600571, abs=5e-9)


def test_log_branch_on_negative_real_axis():
    # physical kinematics WITHOUT deformation at a point where F < 0: lambda -> 0+ limit of ln F is ln|F| - i pi
    wl = qi.massive_box()
    o = Oracle.from_workload(wl, lam=1e-300, eps_order=1)
    sec = o.sector(1)
    F = poly_fn(*sec["F"])
    t = np.array([0.05, 0.05, 0.9])
    Fv = float(F(torch.tensor(t)))
    assert Fv < 0
    U = float(poly_fn(*sec["U"])(torch.tensor(t)))
    c = o.sector_integrand(1, t)
    lam_expected = o.aU1 * np.log(U) + o.aF1 * (np.log(-Fv) - 1j * np.pi)
    assert c[0] == pytest.approx(Fv ** -2, rel=1e-13)
    assert c[1] == pytest.approx(Fv ** -2 * lam_expected, rel=1e-12)


def test_config5_lambda_independence_and_euclidean_limit():
    """Config 5 has no closed form in the container: its VALUE is pinned by invariants only."""
    N, m = 16381, 6
    z = qi.good_vector(N, 5)
    sh = qi.splitmix64_shifts(17, m, 5)
    res = {}
    for lam in (0.3, 0.6):
        o = Oracle.from_workload(qi.nonplanar_vertex(lam=lam))
        S, A, cnt = o.integrate(N, z, sh)
        assert cnt[0] == 0 and cnt[2] == 0
        res[lam] = o.totals(S)
    for k in range(2):
        d = res[0.3][0][k] - res[0.6][0][k]
        assert abs(d.real) <= 4 * np.hypot(res[0.3][1][k].real, res[0.6][1][k].real)
        assert abs(d.imag) <= 4 * np.hypot(res[0.3][1][k].imag, res[0.6][1][k].imag)
    # SURVEY App. B.6 scratch values (context): J_-1 = 0.89835(2) - 1.89262(1) i, J_0 = 5.2397(3) - 0.1113(2) i
    c, e = res[0.3]
    assert abs(c[0] - (0.89835 - 1.89262j)) < 5 * abs(e[0]) + 1e-4
    assert abs(c[1] - (5.2397 - 0.1113j)) < 5 * abs(e[1]) + 1e-3
    # s < 0: Euclidean, Im -> 0 and the deformed result equals the real path
    wl = qi.nonplanar_vertex(s=-5.0)
    oc = Oracle.from_workload(wl, lam=0.3)
    orr = Oracle.from_workload(wl, lam=0.0)
    Sc, _, _ = oc.integrate(N, z, sh)
    Sr, _, _ = orr.integrate(N, z, sh)
    cc, ec = oc.totals(Sc)
    cr, er = orr.totals(Sr)
    for k in range(2):
        assert abs(cc[k].imag) <= 4 * ec[k].imag + 1e-12
        assert abs(cc[k].real - cr[k].real) <= 4 * np.hypot(ec[k].real, er[k].real)


def test_kinematic_scan_points_threshold_and_lambda_independence():
    """points of the paper's s-scan of the one-loop box on the oracle: the imaginary part
    vanishes below the threshold s = 4 M_t^2 = 118336 and is there above it, and the value does not depend
    on lambda (Eq. 14: any deformation that keeps Im F < 0 gives the same integral)."""
    pts = dict((round(s), wl) for s, wl in qi.gghh_box_scan(44))
    N, m = 16381, 6
    z = qi.good_vector(N, 3)
    sh = qi.splitmix64_shifts(11, m, 3)
    res = {}
    for s_phys, lam in ((110000, 0.5), (200000, 0.25), (200000, 0.5)):
        wl = pts[s_phys]
        o = Oracle.from_workload(wl, lam=lam)
        S, A, cnt = o.integrate(N, z, sh)
        assert cnt[0] == 0 and cnt[2] == 0
        res[(s_phys, lam)] = o.totals(S)
    c, e = res[(110000, 0.5)]
    assert abs(c[-1].imag) <= 5 * e[-1].imag + 1e-9 and c[-1].real > 0.3
    (c1, e1), (c2, e2) = res[(200000, 0.25)], res[(200000, 0.5)]
    assert abs((c1[-1] - c2[-1]).real) <= 5 * np.hypot(e1[-1].real, e2[-1].real)
    assert abs((c1[-1] - c2[-1]).imag) <= 5 * np.hypot(e1[-1].imag, e2[-1].imag)
    assert c1[-1].imag > 0.3      # above the threshold s = 4 M_t^2 the integral has an absorptive part
