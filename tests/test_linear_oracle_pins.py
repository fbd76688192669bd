"""Pins of the linear-term oracle (oracle/gx_linear.py) to things other than itself: closed forms,
library quadrature routines the oracle never calls, conservation identities and hand-computed values.
Each test names the passage of PAPER.md ("P:nnn") whose transcription it would catch an error in."""
import math

import numpy as np
import pytest
from numpy.polynomial import hermite_e as HE
from numpy.polynomial import laguerre as LA

from scipy.special import eval_laguerre as special_eval_laguerre, j0 as special_j0, j1 as special_j1

import gx_linear as L
import gx_oracle as O

NX = NY = 16
NAKX, NAKY = 11, 6
DKX, DKY, SHAT = 0.13, 0.1, 0.8


def _geo(Nz, eps=0.18, q=1.4, drifts=True, flat=False):
    z = -math.pi + 2 * math.pi * np.arange(Nz) / Nz
    gradpar = 1.0 / q
    if flat:
        bmag = np.ones(Nz)
        bgrad = np.zeros(Nz)
    else:
        bmag = 1.0 / (1.0 + eps * np.cos(z))
        bgrad = gradpar * eps * np.sin(z) / (1.0 + eps * np.cos(z))          # gradpar d/dz ln B, analytic
    g = dict(bmag=bmag, gds2=1 + (SHAT * z) ** 2, gds21=-SHAT * SHAT * z, gds22=np.full(Nz, SHAT ** 2),
             gbdrift=2 * (np.cos(z) + SHAT * z * np.sin(z)) if drifts else np.zeros(Nz),
             gbdrift0=-2 * SHAT * np.sin(z) if drifts else np.zeros(Nz),
             bgrad=bgrad, jacobian=1.0 / (gradpar * bmag), gradpar=gradpar)
    g["cvdrift"], g["cvdrift0"] = g["gbdrift"].copy(), g["gbdrift0"].copy()
    return g, z


def _rand(shape, seed):
    r = np.random.default_rng(seed)
    return r.standard_normal(shape) + 1j * r.standard_normal(shape)


def _lin(G, Phi, geo, sp, terms, **kw):
    return L.linear_rhs(G, Phi, NX, NY, DKX, DKY, SHAT, geo, [sp], terms=terms, **kw)


def _phi_hermite(m, x):
    """Orthonormal probabilists' Hermite function He_m(x)/sqrt(m!) (library evaluation)."""
    c = np.zeros(m + 1)
    c[m] = 1.0
    return HE.hermeval(x, c) / math.sqrt(math.factorial(m))


# ---------------------------------------------------------------------------- z operators
def test_spectral_z_derivative_closed_form():
    Nz = 16
    z = -math.pi + 2 * math.pi * np.arange(Nz) / Nz
    D, A = L.dz_matrix(Nz), L.abs_kz_matrix(Nz)
    assert np.allclose(D @ np.sin(3 * z), 3 * np.cos(3 * z), atol=1e-12)
    assert np.allclose(D @ np.cos(5 * z), -5 * np.sin(5 * z), atol=1e-12)
    assert np.allclose(D @ np.cos(8 * z), 0, atol=1e-12)                   # Nyquist dropped (reading L2)
    assert np.allclose(D @ np.ones(Nz), 0, atol=1e-13)
    assert np.allclose(A @ np.cos(3 * z), 3 * np.cos(3 * z), atol=1e-12)
    assert np.allclose(A @ np.cos(8 * z), 8 * np.cos(8 * z), atol=1e-12)   # |k_z| keeps it (reading L6)
    assert np.allclose(D, -D.T, atol=1e-13) and np.allclose(A, A.T, atol=1e-13)


# ---------------------------------------------------------------------------- streaming
def test_streaming_matrix_elements_are_hermite_x():
    """-v_t grad_par(sqrt(m+1) H_{m+1} + sqrt(m) H_{m-1}) is -v_t grad_par of 'multiplication by v_par'
    in the orthonormal Hermite basis: <phi_m' | x | phi_m> by Gauss-Hermite quadrature (numpy)."""
    Nz, Nm, kz = 8, 6, 2
    geo, z = _geo(Nz, flat=True, drifts=False)
    sp = dict(Z=1.0, mass=0.5, temp=2.0, dens=1.0, tprim=0, fprim=0, nu_ss=0)       # v_t = 2
    x, w = HE.hermegauss(40)
    w = w / math.sqrt(2 * math.pi)
    X = np.array([[np.sum(w * _phi_hermite(a, x) * x * _phi_hermite(b, x)) for b in range(Nm)] for a in range(Nm)])
    for m0 in range(Nm):
        G = np.zeros((1, Nm, 1, Nz, NAKX, NAKY), complex)
        G[0, m0, 0] = np.exp(1j * kz * z)[:, None, None]
        r = _lin(G, np.zeros((Nz, NAKX, NAKY)), geo, sp, ("stream",))
        for m in range(Nm):
            expect = -2.0 * geo["gradpar"] * 1j * kz * X[m, m0] * G[0, m0, 0]
            assert np.allclose(r[0, m, 0], expect, atol=1e-12), (m0, m)


def test_streaming_of_the_potential_part_of_H():
    """H_{l,0} = G_{l,0} + (Z/tau) J_l Phi (Eq. 4.8): with G = 0 only m = 1 moves, by
    -v_t gradpar i k_z (Z/tau) J_l Phi."""
    Nz, kz = 8, 1
    geo, z = _geo(Nz, flat=True, drifts=False)
    geo = dict(geo, gds2=np.ones(Nz), gds21=np.zeros(Nz))       # z-independent k_perp so that J_l Phi is one harmonic
    sp = dict(Z=2.0, mass=1.0, temp=0.5, dens=1.0, tprim=0, fprim=0, nu_ss=0)
    Phi = np.exp(1j * kz * z)[:, None, None] * _rand((1, NAKX, NAKY), 1)
    r = _lin(np.zeros((1, 3, 2, Nz, NAKX, NAKY)), Phi, geo, sp, ("stream",))
    kx, ky = DKX * O.kx_index(NX), DKY * O.ky_index(NY)
    b = O.kperp2(kx, ky, geo["gds2"], geo["gds21"], geo["gds22"], SHAT) * (0.5 * 1.0 / 4.0)
    vt = math.sqrt(0.5)
    for l in range(2):
        Jl = (-b / 2) ** l / math.factorial(l) * np.exp(-b / 2)
        assert np.allclose(r[0, 1, l], -vt * geo["gradpar"] * 1j * kz * (2.0 / 0.5) * Jl * Phi, atol=1e-12)
    assert np.all(r[0, 0] == 0) and np.all(r[0, 2] == 0)


# ---------------------------------------------------------------------------- streaming + mirror
def test_streaming_plus_mirror_conserve_free_energy_with_jacobian_weight():
    """sum_z (1/B) Re sum_{l,m} conj(H) dH/dt = 0: d/dz of (H_m H_{m+1}/B) integrates to zero.  With
    1/B = 1 + eps cos z and band-limited H the discrete sum is exact; a wrong sign or coefficient in any of
    the four mirror terms (or the stray bracket of P:213 read differently) breaks it."""
    Nz, Nm, Nl = 16, 5, 3
    geo, z = _geo(Nz, drifts=False)
    sp = dict(Z=1.0, mass=1.0, temp=1.0, dens=1.0, tprim=0, fprim=0, nu_ss=0)
    amp = _rand((1, Nm, Nl, 5, NAKX, NAKY), 7)
    G = sum(amp[:, :, :, i, None] * np.exp(1j * kzv * z)[None, None, None, :, None, None]
            for i, kzv in enumerate([-2, -1, 0, 1, 2]))
    Phi0 = np.zeros((Nz, NAKX, NAKY))
    wgt = (1.0 / geo["bmag"])[None, None, None, :, None, None]
    for terms, must_vanish in [(("stream", "mirror"), True), (("stream",), False), (("mirror",), False)]:
        r = _lin(G, Phi0, geo, sp, terms)
        W = np.sum(wgt * np.real(np.conj(G) * r), axis=(1, 2, 3))
        ref = np.sum(np.abs(G) * np.abs(r), axis=(1, 2, 3))
        rel = np.max(np.abs(W) / ref)
        assert (rel < 1e-12) if must_vanish else (rel > 1e-4), (terms, rel)


def test_mirror_hand_values():
    """Mirror force on a single moment (l,m) = (1,1): the four neighbours it feeds and with which weights
    (read off Eq. 4.9 with the roles of source and target exchanged)."""
    Nz = 8
    geo, z = _geo(Nz, drifts=False)
    sp = dict(Z=1.0, mass=1.0, temp=1.0, dens=1.0, tprim=0, fprim=0, nu_ss=0)
    G = np.zeros((1, 3, 3, Nz, NAKX, NAKY), complex)
    src = _rand((Nz, NAKX, NAKY), 3)
    G[0, 1, 1] = src
    r = _lin(G, np.zeros((Nz, NAKX, NAKY)), geo, sp, ("mirror",))
    bg = geo["bgrad"][:, None, None]
    # target (l,m) receives from H_{1,1}:  (l,m)=(1,0): -(l+1)sqrt(m+1) = -2 ; (2,0): -l sqrt(m+1) = -2
    #                                      (1,2): +l sqrt(m) = sqrt2 ; (0,2): +(l+1) sqrt(m) = sqrt2
    assert np.allclose(r[0, 0, 1], -bg * (-2.0) * src)
    assert np.allclose(r[0, 0, 2], -bg * (-2.0) * src)
    assert np.allclose(r[0, 2, 1], -bg * math.sqrt(2.0) * src)
    assert np.allclose(r[0, 2, 0], -bg * math.sqrt(2.0) * src)
    touched = {(0, 1), (0, 2), (2, 1), (2, 0)}
    for m in range(3):
        for l in range(3):
            if (m, l) not in touched:
                assert np.all(r[0, m, l] == 0)


# ---------------------------------------------------------------------------- drifts
def test_drift_matrix_elements_by_library_quadrature():
    """grad-B term = multiplication by mu B in the psi_l basis, curvature term = multiplication by v_par^2
    in the Hermite basis: matrix elements by Gauss-Laguerre / Gauss-Hermite quadrature (numpy)."""
    Nz, Nm, Nl = 4, 5, 4
    geo, z = _geo(Nz, flat=True)
    sp = dict(Z=-1.0, mass=1.0, temp=2.0, dens=1.0, tprim=0, fprim=0, nu_ss=0)
    tz = 2.0 / -1.0
    kx, ky = DKX * O.kx_index(NX), DKY * O.ky_index(NY)
    wk, wb = L.drift_frequencies(kx, ky, geo, SHAT)
    xl, wl = LA.laggauss(30)
    psi = lambda l, x: (-1.0) ** l * LA.lagval(x, np.eye(l + 1)[l])
    ML = np.array([[np.sum(wl * psi(a, xl) * xl * psi(b, xl)) for b in range(Nl)] for a in range(Nl)])
    xh, wh = HE.hermegauss(40)
    wh = wh / math.sqrt(2 * math.pi)
    MH = np.array([[np.sum(wh * _phi_hermite(a, xh) * xh ** 2 * _phi_hermite(b, xh)) for b in range(Nm)]
                   for a in range(Nm)])
    G = _rand((1, Nm, Nl, Nz, NAKX, NAKY), 11)
    geo_b = dict(geo, cvdrift=np.zeros(Nz), cvdrift0=np.zeros(Nz))
    geo_k = dict(geo, gbdrift=np.zeros(Nz), gbdrift0=np.zeros(Nz))
    rb = _lin(G, np.zeros((Nz, NAKX, NAKY)), geo_b, sp, ("drift",))
    rk = _lin(G, np.zeros((Nz, NAKX, NAKY)), geo_k, sp, ("drift",))
    assert np.allclose(rb[0], -1j * tz * wb * np.einsum("ab,mbzxy->mazxy", ML, G[0]), atol=1e-11)
    assert np.allclose(rk[0], -1j * tz * wk * np.einsum("ab,blzxy->alzxy", MH, G[0]), atol=1e-11)
    # s-alpha closed form of the frequencies (reading L3): w_d = ky (cos z + shat z sin z) - kx sin z
    zz = z[:, None, None]
    assert np.allclose(wb, ky[None, None, :] * (np.cos(zz) + SHAT * zz * np.sin(zz)) - kx[None, :, None] * np.sin(zz))
    # anti-Hermitian: no free-energy change, mode by mode
    r = _lin(G, np.zeros((Nz, NAKX, NAKY)), geo, sp, ("drift",))
    assert np.max(np.abs(np.sum(np.real(np.conj(G) * r), axis=(1, 2)))) < 1e-11


# ---------------------------------------------------------------------------- drive
def test_drive_hand_values_at_zero_larmor_radius():
    Nz = 4
    geo, z = _geo(Nz, flat=True)
    sp = dict(Z=1.0, mass=1e-30, temp=1.0, dens=1.0, tprim=6.9, fprim=2.2, nu_ss=0)      # b = 0: J_0 = 1
    Phi = _rand((Nz, NAKX, NAKY), 5)
    r = _lin(np.zeros((1, 4, 3, Nz, NAKX, NAKY)), Phi, geo, sp, ("drive",))
    iky = 1j * (DKY * O.ky_index(NY))[None, None, :]
    assert np.allclose(r[0, 0, 0], iky * 2.2 * Phi)                 # density gradient drives density
    assert np.allclose(r[0, 0, 1], iky * 6.9 * Phi)                 # temperature gradient drives T_perp
    assert np.allclose(r[0, 2, 0], iky * 6.9 * Phi / math.sqrt(2))  # ... and T_par
    for (m, l) in [(0, 2), (1, 0), (1, 1), (2, 1), (3, 0)]:
        assert np.max(np.abs(r[0, m, l])) < 1e-25          # b = O(1e-30), not exactly 0


# ---------------------------------------------------------------------------- Dougherty
def test_dougherty_conserves_density_momentum_energy_and_damps_the_rest():
    Nz, Nm, Nl = 4, 5, 3
    geo, z = _geo(Nz, flat=True)
    nu = 0.37
    sp = dict(Z=1.0, mass=1.0, temp=1.0, dens=1.0, tprim=0, fprim=0, nu_ss=nu)
    G = _rand((1, Nm, Nl, Nz, NAKX, NAKY), 13)
    r = _lin(G, np.zeros((Nz, NAKX, NAKY)), geo, sp, ("coll",))
    k0 = (slice(None), 0, 0)                                   # kx = ky = 0: b = 0
    s = np.max(np.abs(G))
    assert np.max(np.abs(r[0, 0, 0][k0])) < 1e-13 * s          # density
    assert np.max(np.abs(r[0, 1, 0][k0])) < 1e-13 * s          # parallel momentum
    assert np.max(np.abs(math.sqrt(2) * r[0, 2, 0][k0] + 2 * r[0, 0, 1][k0])) < 1e-12 * s   # T_par + 2 T_perp
    assert np.allclose(r[0, 3, 1][k0], -nu * (2 * 1 + 3) * G[0, 3, 1][k0])                 # plain damping
    assert np.allclose(r[0, 4, 2][k0], -nu * (2 * 2 + 4) * G[0, 4, 2][k0])
    # finite b: the rate of a moment outside the conserved set is -nu (b + 2l + m)
    kx, ky = DKX * O.kx_index(NX), DKY * O.ky_index(NY)
    b = O.kperp2(kx, ky, geo["gds2"], geo["gds21"], geo["gds22"], SHAT)
    assert np.allclose(r[0, 4, 1], -nu * (b + 2 + 4) * G[0, 4, 1])
    # free energy never grows under like-particle collisions
    assert np.all(np.sum(np.real(np.conj(G) * r), axis=(1, 2)) <= 1e-12)


def _velocity_space_quadrature(nt=60, nv=40):
    """Library quadrature in (mu B, v_par): d^3v F_M -> sum over (t_i, v_j) with weights wt_i wv_j, where
    int_0^inf e^-t dt and int e^{-v^2/2}/sqrt(2 pi) dv are the two measures (Eq. 2.2; Eq. 4.1)."""
    t, wt = LA.laggauss(nt)
    v, wv = HE.hermegauss(nv)
    return t, wt, v, wv / math.sqrt(2 * math.pi)


def _finite_b_setup(Nl, Nm, seed):
    """Two z points with B != 1, a species with Z, m, tau != 1, b_s between 0 and ~0.25 over the modes."""
    Nz = 2
    geo = dict(bmag=np.array([1.0, 1.3]), gds2=np.array([1.1, 0.8]), gds21=np.array([0.15, -0.2]),
               gds22=np.array([0.64, 0.9]), gbdrift=np.zeros(Nz), gbdrift0=np.zeros(Nz), cvdrift=np.zeros(Nz),
               cvdrift0=np.zeros(Nz), bgrad=np.zeros(Nz), jacobian=np.array([1.0, 1.0 / 1.3]), gradpar=0.7)
    Zs, ms, ts = 2.0, 1.5, 0.8
    kx, ky = DKX * O.kx_index(NX), DKY * O.ky_index(NY)
    kxx, kyy = kx[None, :, None], ky[None, None, :]
    kp2 = (kyy ** 2 * geo["gds2"][:, None, None] + 2 * kxx * kyy * geo["gds21"][:, None, None] / SHAT
           + kxx ** 2 * geo["gds22"][:, None, None] / SHAT ** 2)
    b = kp2 * ts * ms / (Zs ** 2 * geo["bmag"][:, None, None] ** 2)          # P:85, by hand
    G = _rand((1, Nm, Nl, Nz, NAKX, NAKY), seed)
    Phi = _rand((Nz, NAKX, NAKY), seed + 1)
    # H_{l,m} = G_{l,m} + (Z/tau) J_l Phi delta_m0 (Eq. 4.8), J_l typed out from Eq. 4.7
    H = G[0].copy()
    for l in range(Nl):
        H[0, l] += (Zs / ts) * ((-b / 2) ** l / math.factorial(l) * np.exp(-b / 2)) * Phi
    return geo, (Zs, ms, ts), b, G, Phi, H, ky


def test_dougherty_field_particle_terms_from_the_velocity_space_operator_at_finite_b():
    """Eq. 2.5-2.8 evaluated in velocity space by library Gauss-Laguerre x Gauss-Hermite quadrature
    and projected with Eq. 4.1: the field-particle moments u_par, u_perp, T_par, T_perp (Eq. 4.14-4.17,
    P:251-258) of h = sum_{l,m} H_{l,m} psi_l phi_m F_M and the Laguerre-Hermite transform of
    ( T [(v^2-1) + 2(muB-1)] J0 + u_par v J0 + u_perp v_perp J1 ) F_M, at finite b, Phi != 0, B != 1.
    Nl = 6 and b <= 0.25 keep the one difference -- the paper sets J_l = 0 for l >= Nl, the integral
    does not -- below 1e-6.  A wrong sign, power of b, index shift or H<->G in Eq. 4.13-4.17 fails."""
    Nl, Nm, nu = 6, 4, 0.37
    geo, (Zs, ms, ts), b, G, Phi, H, _ = _finite_b_setup(Nl, Nm, 41)
    assert 0.2 < b.max() < 0.3
    sp = dict(Z=Zs, mass=ms, temp=ts, dens=1.0, tprim=0, fprim=0, nu_ss=nu)
    r = _lin(G, Phi, geo, sp, ("coll",))[0]                                  # [m][l][z][kx][ky]
    t, wt, v, wv = _velocity_space_quadrature()
    psi = np.array([(-1.0) ** l * special_eval_laguerre(l, t) for l in range(Nl)])      # [l][t]
    phi = np.array([_phi_hermite(m, v) for m in range(Nm)])                              # [m][v]
    alpha = np.sqrt(2.0 * t[None, None, None, :] * b[..., None])                         # [z][kx][ky][t]
    J0, J1 = special_j0(alpha), special_j1(alpha)
    vperp = np.sqrt(2.0 * t)
    # hhat(t, v) = sum H_{l,m} psi_l(t) phi_m(v): h = hhat F_M
    hhat = np.einsum("mlzxy,lt,mv->zxytv", H, psi, phi)
    W = wt[:, None] * wv[None, :]                                                        # [t][v]
    upar = np.einsum("zxytv,zxyt,v,tv->zxy", hhat, J0, v, W)
    uperp = np.einsum("zxytv,zxyt,t,tv->zxy", hhat, J1, vperp, W)
    Tpar = np.einsum("zxytv,zxyt,v,tv->zxy", hhat, J0, v ** 2 - 1, W)
    Tperp = np.einsum("zxytv,zxyt,t,tv->zxy", hhat, J0, t - 1, W)
    Tbar = (Tpar + 2 * Tperp) / 3                                                        # Eq. 2.8 / 4.18
    one_t, one_v = np.ones_like(t), np.ones_like(v)
    bracket = (Tbar[..., None, None] * ((v ** 2 - 1)[None, :] * one_t[:, None] + 2 * (t - 1)[:, None] * one_v[None, :])
               * J0[..., None]
               + upar[..., None, None] * v[None, :] * J0[..., None]
               + uperp[..., None, None] * (vperp[:, None] * one_v[None, :]) * J1[..., None])          # [z][kx][ky][t][v]
    FP = np.einsum("zxytv,lt,mv,tv->mlzxy", bracket, psi, phi, W)
    expect = np.empty_like(r)
    for m in range(Nm):
        for l in range(Nl):
            expect[m, l] = -nu * (b + 2 * l + m) * H[m, l] + nu * FP[m, l]
    scale = np.max(np.abs(expect))
    assert np.max(np.abs(r - expect)) < 2e-6 * scale
    # the field-particle part is not small: without it the comparison fails by O(1e-2)
    assert np.max(np.abs(nu * FP[:3])) > 1e-2 * scale
    # and it only reaches m = 0, 1, 2
    assert np.max(np.abs(FP[3])) < 1e-12 * scale


def test_drive_terms_at_finite_larmor_radius_from_the_maxwellian_gradient():
    """Eq. 4.12, Phi parts: the drive is i w_* <J0 Phi> [1/L_n + (E - 3/2)/L_T] F_M with
    E = v^2/2 + muB (grad F_M at constant energy, Eq. 2.1-2.2), transformed with Eq. 4.1:
    D_{l,0} = i ky Phi int psi_l J0 [fprim + tprim (t - 1)] e^-t dt,  D_{l,2} = i ky Phi tprim/sqrt2 int psi_l J0 e^-t dt,
    by library Gauss-Laguerre quadrature at finite b (the b = 0 hand values are a separate test)."""
    Nl, Nm = 6, 4
    geo, (Zs, ms, ts), b, G, Phi, H, ky = _finite_b_setup(Nl, Nm, 43)
    sp = dict(Z=Zs, mass=ms, temp=ts, dens=1.0, tprim=6.9, fprim=2.2, nu_ss=0)
    r = _lin(np.zeros_like(G), Phi, geo, sp, ("drive",))[0]
    t, wt, v, wv = _velocity_space_quadrature()
    J0 = special_j0(np.sqrt(2.0 * t[None, None, None, :] * b[..., None]))
    iky = 1j * ky[None, None, :]
    s0 = np.max(np.abs(6.9 * iky * Phi))
    for l in range(Nl):
        psi_l = (-1.0) ** l * special_eval_laguerre(l, t)
        d0 = np.einsum("zxyt,t->zxy", J0, wt * psi_l * (2.2 + 6.9 * (t - 1.0)))
        d2 = np.einsum("zxyt,t->zxy", J0, wt * psi_l) * 6.9 / math.sqrt(2.0)
        assert np.max(np.abs(r[0, l] - iky * d0 * Phi)) < 2e-6 * s0, l
        assert np.max(np.abs(r[2, l] - iky * d2 * Phi)) < 2e-6 * s0, l
        assert np.all(r[1, l] == 0) and np.all(r[3, l] == 0)
    assert np.max(np.abs(r[0, 1])) > 0.05 * s0 and np.max(np.abs(r[0, 2])) > 1e-3 * s0       # finite-b parts are visible


def test_curvature_drift_frequency_with_a_pressure_term():
    """w_d^kappa = (ky cvdrift + kx cvdrift0/shat)/2 (reading L3; Eq. E10-E11) with cvdrift != gbdrift:
    s-alpha arrays plus a constant pressure-gradient part c0 in cvdrift  =>
    w_d^kappa = ky (cos z + shat z sin z + c0/2) - kx sin z, w_d^gradB without c0; and the curvature term of
    Eq. 4.9 is -i (tau/Z) w_d^kappa <phi_m'| v^2 |phi_m> H (Gauss-Hermite matrix elements)."""
    Nz, Nm, Nl, c0 = 4, 5, 2, 0.6
    geo, z = _geo(Nz, flat=True)
    geo = dict(geo, cvdrift=geo["gbdrift"] + c0)
    kx, ky = DKX * O.kx_index(NX), DKY * O.ky_index(NY)
    zz = z[:, None, None]
    wk_hand = ky[None, None, :] * (np.cos(zz) + SHAT * zz * np.sin(zz) + c0 / 2) - kx[None, :, None] * np.sin(zz)
    wb_hand = ky[None, None, :] * (np.cos(zz) + SHAT * zz * np.sin(zz)) - kx[None, :, None] * np.sin(zz)
    wk, wb = L.drift_frequencies(kx, ky, geo, SHAT)
    assert np.allclose(wk, wk_hand, atol=1e-14) and np.allclose(wb, wb_hand, atol=1e-14)
    sp = dict(Z=-1.0, mass=1.0, temp=2.0, dens=1.0, tprim=0, fprim=0, nu_ss=0)
    G = _rand((1, Nm, Nl, Nz, NAKX, NAKY), 47)
    xh, wh = HE.hermegauss(40)
    wh = wh / math.sqrt(2 * math.pi)
    MH = np.array([[np.sum(wh * _phi_hermite(a, xh) * xh ** 2 * _phi_hermite(c, xh)) for c in range(Nm)]
                   for a in range(Nm)])
    geo_k = dict(geo, gbdrift=np.zeros(Nz), gbdrift0=np.zeros(Nz))
    rk = _lin(G, np.zeros((Nz, NAKX, NAKY)), geo_k, sp, ("drift",))
    assert np.allclose(rk[0], -1j * (2.0 / -1.0) * wk_hand * np.einsum("ab,blzxy->alzxy", MH, G[0]), atol=1e-11)


# ---------------------------------------------------------------------------- hyper-dissipation
def test_hyper_dissipation_closed_forms():
    Nz, Nm = 8, 6
    geo, z = _geo(Nz)
    sp = dict(Z=1.0, mass=1.0, temp=4.0, dens=1.0, tprim=0, fprim=0, nu_ss=0)          # v_t = 2
    G = _rand((1, Nm, 1, Nz, NAKX, NAKY), 17)
    r = _lin(G, np.zeros((Nz, NAKX, NAKY)), geo, sp, ("hypervisc",), D_hyper=0.05, n_hyper=4)
    kx, ky = DKX * O.kx_index(NX), DKY * O.ky_index(NY)
    kp2 = (kx[None, :, None] - SHAT * z[:, None, None] * ky[None, None, :]) ** 2 + ky[None, None, :] ** 2
    rate = r[0, 2, 0] / G[0, 2, 0]
    assert np.allclose(rate, -0.05 * (kp2 / kp2.max()) ** 4, atol=1e-13)
    assert abs(rate.real.min() + 0.05) < 1e-13 and np.all(rate[:, 0, 0] == 0)
    kz = 3
    G2 = np.zeros_like(G)
    for m in range(Nm):
        G2[0, m, 0] = np.exp(1j * kz * z)[:, None, None] * (m + 1)
    r2 = _lin(G2, np.zeros((Nz, NAKX, NAKY)), geo, sp, ("hypercoll",), f_hyp=1.0)
    p = Nm / 2
    nuhyp = 2.5 * (p + 0.5) / (Nm - 1) ** (p + 0.5) * (geo["gradpar"] * kz) * 2.0
    for m in range(Nm):
        expect = -nuhyp * m ** p * G2[0, m, 0] if m > 2 else 0 * G2[0, m, 0]
        assert np.allclose(r2[0, m, 0], expect, atol=1e-12), m


# ---------------------------------------------------------------------------- time stepping
def test_ssp_rk3_is_third_order_taylor_on_linear_problem():
    lam, dt = -0.7 + 2.0j, 0.1
    y = L.ssp_rk3_step(1.0 + 0j, dt, lambda v: lam * v)
    x = lam * dt
    assert abs(y - (1 + x + x * x / 2 + x ** 3 / 6)) < 1e-15
    errs = []
    for n in (20, 40):
        v = 1.0 + 0j
        for _ in range(n):
            v = L.ssp_rk3_step(v, 1.0 / n, lambda u: lam * u)
        errs.append(abs(v - np.exp(lam)))
    assert 6.5 < errs[0] / errs[1] < 9.5                      # third order: error ratio ~ 8


def test_full_rhs_is_sum_of_parts_and_linear_in_g_without_bracket():
    Nz = 4
    geo, z = _geo(Nz)
    sp = dict(Z=1.0, mass=1.0, temp=1.0, dens=1.0, tprim=6.9, fprim=2.2, nu_ss=0.01)
    G = 1e-3 * _rand((1, 4, 2, Nz, NAKX, NAKY), 19)
    K = (NAKX - 1) // 2
    G[..., 0, 0] = 0
    G[..., NAKX - 1:K:-1, 0] = np.conj(G[..., 1:K + 1, 0])
    full = L.rhs(G, NX, NY, DKX, DKY, SHAT, geo, [sp])
    lin = L.rhs(G, NX, NY, DKX, DKY, SHAT, geo, [sp], nonlinear=False)
    Phi = O.field_solve(G, NX, NY, DKX, DKY, SHAT, geo, [sp])
    nl = O.nonlinear_rhs(G, Phi, NX, NY, DKX, DKY, SHAT, geo, [sp], method="conv_np")
    assert np.allclose(full, lin + nl, atol=1e-14)
    assert np.allclose(L.rhs(2 * G, NX, NY, DKX, DKY, SHAT, geo, [sp], nonlinear=False), 2 * lin, atol=1e-15)


# ---------------------------------------------------------------------------- twist-and-shift linking
def test_twist_shift_chains_partition_the_modes_and_keep_kperp_continuous():
    Nx, Ny, shat, dky = 192, 64, 0.8, 0.1
    jt = max(1, round(2 * math.pi * shat))
    dkx = 2 * math.pi * shat * dky / jt
    assert L.jtwist_of(dkx, dky, shat) == 5 and L.jtwist_of(dkx, dky, -shat) == -5
    with pytest.raises(ValueError):
        L.jtwist_of(1.07 * dkx, dky, shat)
    chains = L.twist_shift_chains(Nx, Ny, 5)
    seen = sorted((i, q) for q, rows in chains for i in rows)
    assert seen == sorted((i, q) for i in range(127) for q in range(22))          # every mode exactly once
    assert sorted(len(r) for q, r in chains if q == 1) == [25, 25, 25, 26, 26]       # 127 modes in 5 classes mod 5
    assert all(len(r) == 1 for q, r in chains if q == 0)
    kxi = O.kx_index(Nx)
    z = np.linspace(-math.pi, math.pi, 7)
    for q, rows in chains:
        for a, b in zip(rows[:-1], rows[1:]):
            kxa, kxb, ky = dkx * kxi[a], dkx * kxi[b], dky * q
            # Eq. 4.29: H(kx,ky,z) = H(kx + dk,ky,z + 2 pi): the s-alpha k_perp^2 = (kx - shat z ky)^2 + ky^2 must agree
            assert np.allclose((kxa - shat * z * ky) ** 2, (kxb - shat * (z + 2 * math.pi) * ky) ** 2, atol=1e-12)


def test_linked_z_operators_closed_form_on_a_ballooning_harmonic():
    Nz, jt, gradpar = 8, 2, 0.7
    chains = L.twist_shift_chains(NX, NY, jt)
    q, rows = max(chains, key=lambda c: len(c[1]))
    Lc = len(rows)
    assert Lc >= 3
    z = -math.pi + 2 * math.pi * np.arange(Nz) / Nz
    for jmode in (1, -2, 5):
        kap = jmode / Lc
        f = np.zeros((Nz, NAKX, NAKY), complex)
        for n, i in enumerate(rows):
            f[:, i, q] = np.exp(1j * kap * (z - 2 * math.pi * n))        # mode n holds Psi(theta = z - 2 pi n)
        d = L.apply_z_operator(f, "d", gradpar, NX, NY, "linked", jt)
        a = L.apply_z_operator(f, "a", gradpar, NX, NY, "linked", jt)
        assert np.allclose(d, 1j * kap * gradpar * f, atol=1e-12)
        assert np.allclose(a, abs(kap) * gradpar * f, atol=1e-12)
    # ky = 0 (and every unlinked mode) keeps the plain periodic operator; the operator stays anti-symmetric
    g = _rand((Nz, NAKX, NAKY), 23)
    dl = L.apply_z_operator(g, "d", gradpar, NX, NY, "linked", jt)
    dp = L.apply_z_operator(g, "d", gradpar, NX, NY, "periodic")
    assert np.allclose(dl[:, :, 0], dp[:, :, 0], atol=1e-13)
    assert not np.allclose(dl[:, :, 1], dp[:, :, 1], atol=1e-3)
    assert abs(np.sum(np.real(np.conj(g) * dl))) < 1e-11 * np.sum(np.abs(g) ** 2)


def test_linked_rhs_differs_only_through_the_z_operators():
    Nz = 4
    geo, z = _geo(Nz)
    dkx = 2 * math.pi * SHAT * DKY / 5
    sp = dict(Z=1.0, mass=1.0, temp=1.0, dens=1.0, tprim=6.9, fprim=2.2, nu_ss=0.01)
    G = _rand((1, 5, 2, Nz, NAKX, NAKY), 29)
    Phi = _rand((Nz, NAKX, NAKY), 31)
    kw = dict(Nx=NX, Ny=NY, dkx=dkx, dky=DKY, shat=SHAT, geo=geo, species=[sp])
    a = L.linear_rhs(G, Phi, boundary="linked", **kw)
    b = L.linear_rhs(G, Phi, boundary="periodic", **kw)
    local = ("mirror", "drift", "drive", "coll", "hypervisc")
    assert np.allclose(L.linear_rhs(G, Phi, boundary="linked", terms=local, **kw),
                       L.linear_rhs(G, Phi, boundary="periodic", terms=local, **kw), atol=0)
    assert np.allclose(a[..., 0], b[..., 0], atol=1e-12) and not np.allclose(a[..., 1:], b[..., 1:], atol=1e-3)


# ---------------------------------------------------------------------------- end-damping layer (Eq. 4.30)
def test_end_damping_profile_hand_values_and_structure():
    """d(zh) = A [1 - 2 zh^2/(1 + zh^4)], |zh| < 1, distance from either end of the extended domain in units of
    L_z/8; ky = 0 untouched.  Periodic domains (L = 1), Nz = 16: z_width = 2 pi/8 = two grid steps."""
    A, Nz = 0.7, 16
    d = L.end_damping_profile(Nz, NX, NY, A, 0.125, "periodic")
    f = lambda zh: A * (1 - 2 * zh ** 2 / (1 + zh ** 4))
    expect = np.zeros(Nz)
    expect[0] = f(0.0)             # z_0 = -pi is the lower end itself: d = A
    expect[1] = f(0.5)             # one step = half a width from the lower end: A (1 - 0.5/1.0625)
    expect[15] = f(0.5)            # one step below the upper end (theta = pi is not a grid point)
    assert abs(f(0.5) - A * (1 - 0.5 / 1.0625)) < 1e-15 and abs(f(1.0)) < 1e-15
    for i in range(NAKX):
        for q in range(1, NAKY):
            assert np.allclose(d[:, i, q], expect, atol=1e-15)
    assert np.all(d[:, :, 0] == 0)                     # zonal modes are not filtered
    # linked domains: only the two end segments of a chain are damped, symmetrically, and the width grows with L
    jt = 2
    dl = L.end_damping_profile(Nz, NX, NY, A, 0.125, "linked", jt)
    z = -math.pi + 2 * math.pi * np.arange(Nz) / Nz
    for q, rows in L.twist_shift_chains(NX, NY, jt):
        if q == 0:
            continue
        Lc = len(rows)
        theta = np.concatenate([z - 2 * math.pi * n for n in range(Lc - 1, -1, -1)])       # increasing ballooning angle
        prof = np.concatenate([dl[:, rows[n], q] for n in range(Lc - 1, -1, -1)])
        lo, hi, w = -math.pi - 2 * math.pi * (Lc - 1), math.pi, 2 * math.pi * Lc / 8
        ref = np.where(theta - lo < w, f((theta - lo) / w), 0.0) + np.where(hi - theta < w, f((hi - theta) / w), 0.0)
        assert np.allclose(prof, ref, atol=1e-14)
        assert np.all(prof >= 0) and prof[0] == A and np.all(prof[(theta - lo >= w) & (hi - theta >= w)] == 0)
        # reflection symmetry about the middle of the extended domain (the end point theta_hi is off-grid by one step)
        assert np.allclose(prof[1:], prof[1:][::-1], atol=1e-14)


def test_end_damping_acts_on_H_for_nonzonal_modes_only():
    Nz = 8
    geo, z = _geo(Nz)
    sp = dict(Z=2.0, mass=1.0, temp=0.5, dens=1.0, tprim=0, fprim=0, nu_ss=0)
    G = _rand((1, 3, 2, Nz, NAKX, NAKY), 53)
    Phi = _rand((Nz, NAKX, NAKY), 54)
    dmp = dict(A=0.3, width_frac=0.25)
    r = L.linear_rhs(G, Phi, NX, NY, DKX, DKY, SHAT, geo, [sp], terms=(), damping=dmp)
    d = L.end_damping_profile(Nz, NX, NY, 0.3, 0.25)
    kx, ky = DKX * O.kx_index(NX), DKY * O.ky_index(NY)
    b = O.kperp2(kx, ky, geo["gds2"], geo["gds21"], geo["gds22"], SHAT) * (0.5 * 1.0 / 4.0) / geo["bmag"][:, None, None] ** 2
    for l in range(2):
        Jl = (-b / 2) ** l / math.factorial(l) * np.exp(-b / 2)
        assert np.allclose(r[0, 0, l], -d * (G[0, 0, l] + (2.0 / 0.5) * Jl * Phi), atol=1e-13)     # m = 0: H = G + (Z/tau) J_l Phi
        assert np.allclose(r[0, 2, l], -d * G[0, 2, l], atol=1e-13)
    assert np.all(r[..., 0] == 0) and np.max(np.abs(r[..., 1:])) > 0.01
    # without the option nothing changes
    assert np.all(L.linear_rhs(G, Phi, NX, NY, DKX, DKY, SHAT, geo, [sp], terms=()) == 0)
