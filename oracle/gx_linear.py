"""fp64 CPU oracle for the linear terms of the Fourier-Laguerre-Hermite gyrokinetic system and for
the full right-hand side / SSP-RK3 step (arxiv 2209.06731 "GX", electrostatic limit).
TEST INFRASTRUCTURE ONLY: only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s CPU legs may
import this file.  It shares no code with the CUDA path and imports only its sibling ``gx_oracle``.

"P:nnn" = PAPER.md line nnn.  beta_ref = 0, so A_par = dB_par = 0 and (Eq. 4.8)

    H_{l,m} = G_{l,m} + (Z_s/tau_s) J_l Phi delta_{m0},      J_l = (1/l!)(-b_s/2)^l e^{-b_s/2}  (Eq. 4.7)

with H, G, J == 0 outside 0 <= l < Nl, 0 <= m < Nm (closure by truncation P:305).
``linear_rhs`` returns dG/dt without the nonlinear term, i.e. Eq. 4.9 solved for dG/dt:

    - v_ts grad_par( sqrt(m+1) H_{l,m+1} + sqrt(m) H_{l,m-1} )                                   streaming
    - v_ts (grad_par ln B) [ -(l+1) sqrt(m+1) H_{l,m+1} - l sqrt(m+1) H_{l-1,m+1}
                             + l sqrt(m) H_{l,m-1} + (l+1) sqrt(m) H_{l+1,m-1} ]                 mirror
    - i (tau_s/Z_s) w_d^kappa [ sqrt((m+1)(m+2)) H_{l,m+2} + (2m+1) H_{l,m} + sqrt(m(m-1)) H_{l,m-2} ]
    - i (tau_s/Z_s) w_d^gradB [ (l+1) H_{l+1,m} + (2l+1) H_{l,m} + l H_{l-1,m} ]                 drifts
    + D_{l,m}                                     Eq. 4.12, Phi parts only
    + C_{l,m}                                     Eq. 4.13-4.18, Dougherty
    - D (kperp2/kperp2_max)^n G_{l,m}             Eq. 4.26
    - nu_hyp m^p G_{l,m}  (m > 2)                 Eq. 4.27-4.28

Readings of silent / garbled points (rows L1-L8):
  L1  the stray "]" on P:213 is a garble: all four mirror terms multiply grad_par ln B.
  L2  grad_par = gradpar * d/dz with constant gradpar, d/dz spectral on the periodic grid
      z_i = -pi + 2 pi i/Nz (k_z integer); the Nyquist mode's derivative is zero.  boundary="periodic":
      each (kx,ky) is periodic by itself (SURVEY App. A "first implementation").  boundary="linked": the
      twist-and-shift condition of P:322-327, H(kx,ky,z) = H(kx + dk, ky, z + 2 pi), dk = 2 pi ky shat: the
      modes kx_0 + n dk (n integer, inside the dealiased set) of one ky form ONE periodic extended domain of
      L 2 pi, on which mode n holds the segment theta = z - 2 pi n of the ballooning function; the z operators
      are spectral on that domain (k = j/L, Nyquist dropped in the derivative).  dk is a whole number
      jtwist*q of kx grid steps because Lx/Ly = jtwist/(2 pi |shat|).
  L9  end-damping layer Eq. 4.30, optional (``damping=dict(A=..., width_frac=1/8)``): distance
      measured from BOTH ends of each extended domain, z_width = L_z/8 with L_z the length of that domain, acts
      on H, non-zonal modes only; A is a free parameter (the paper uses 0.1/dt).
  L3  w_d^gradB = (ky gbdrift + kx gbdrift0/shat)/2, w_d^kappa = (ky cvdrift + kx cvdrift0/shat)/2
      (P:229 with Eq. E9-E11: the arrays carry a factor 2 and gbdrift0 a factor shat).
  L4  i w_* = i ky; 1/L_n = fprim, 1/L_T = tprim.
  L5  k_perp,max^2 = max over all z and kept (kx,ky) of kperp2 ("largest dealiased perpendicular
      wavenumber in the simulation"); D = 0.05, n = 4 default (P:303's "n = 2" differs).
  L6  hyper-collisions: p = Nm/2, m_max = Nm - 1, |k_par| = gradpar |k_z| applied spectrally in z
      (Nyquist kept at Nz/2), f_hyp = 1.
  L7  "b" without subscript on P:246 is b_s; sums printed to N_l run over l < Nl.
  L8  SSP-RK3 in Shu-Osher form (the paper cites Gottlieb et al.).

Pins (tests/test_linear_oracle_pins.py): spectral derivative of a single harmonic; Hermite-ladder
streaming eigenvalues = Gauss-Hermite nodes; drift matrices' eigenvalues = Gauss-Laguerre nodes and
squared Gauss-Hermite nodes (library quadrature routines the oracle does not call); 1/B-weighted
free-energy identity of streaming + mirror; anti-Hermiticity of the drift terms; Dougherty conservation of
density, momentum and energy at k_perp = 0 and its damping rates; hand values of the drive; closed forms
of both hyper-dissipation terms; SSP-RK3 order on dy/dt = lambda y.  Finite Larmor radius: every coefficient
of the Dougherty field-particle terms (Eq. 4.13-4.17) against the velocity-space operator Eq. 2.5-2.8 by
library Gauss-Laguerre x Gauss-Hermite quadrature at b up to 0.25, Phi != 0, B != 1, Z, m, tau != 1; the
drive's 1/L_n and 1/L_T brackets at finite b against the Maxwellian-gradient integrals; w_d^kappa with
cvdrift != gbdrift against the s-alpha closed form.
"""
from __future__ import annotations

import math

import numpy as np

import gx_oracle as O


def _get(sp, k):
    if isinstance(sp, dict):
        return sp[k]
    return getattr(sp, k)


def _nu(sp):
    if isinstance(sp, dict):
        return sp.get("nu_ss", sp.get("nu", 0.0))
    return getattr(sp, "nu_ss", 0.0)


# ============================================================================ z operators
def kz_index(Nz):
    """Integer k_z of the length-Nz DFT in storage order 0,1,..,-1."""
    return np.array([k if k <= Nz // 2 else k - Nz for k in range(Nz)], dtype=np.float64)


def dz_matrix(Nz):
    """D[z][z'] of the spectral d/dz on the periodic grid of length 2 pi (Eq. 4.10-4.11):
    F^-1 diag(i k_z) F written as an explicit real matrix; the Nyquist mode is dropped (reading L2)."""
    k = kz_index(Nz)
    if Nz % 2 == 0:
        k[Nz // 2] = 0.0
    z = np.arange(Nz)
    ph = np.exp(2j * math.pi * np.outer(z, np.arange(Nz)) / Nz)          # e^{+i 2 pi z k / Nz}
    return np.real((ph * (1j * k)[None, :]) @ np.conj(ph).T) / Nz


def abs_kz_matrix(Nz):
    """A[z][z'] of the spectral |k_z| (Eq. 4.28's |k_par| without gradpar; reading L6)."""
    k = np.abs(kz_index(Nz))
    z = np.arange(Nz)
    ph = np.exp(2j * math.pi * np.outer(z, np.arange(Nz)) / Nz)
    return np.real((ph * k[None, :]) @ np.conj(ph).T) / Nz


def ext_operator_matrices(Nz, L):
    """(d/dzeta, |k_zeta|) on the periodic extended domain of L segments of Nz points (length 2 pi L):
    explicit DFT sums with k = j/L; the Nyquist mode is dropped in the derivative (reading L2)."""
    N = Nz * L
    j = np.array([q if q <= N // 2 else q - N for q in range(N)], dtype=np.float64)
    kd = j / L
    if N % 2 == 0:
        kd = kd.copy()
        kd[N // 2] = 0.0
    ph = np.exp(2j * math.pi * np.outer(np.arange(N), np.arange(N)) / N)
    D = np.real((ph * (1j * kd)[None, :]) @ np.conj(ph).T) / N
    A = np.real((ph * (np.abs(j) / L)[None, :]) @ np.conj(ph).T) / N
    return D, A


def twist_shift_chains(Nx, Ny, jtwist):
    """Linked chains of the compact modes under H(kx,ky,z) = H(kx + dk,ky,z + 2 pi) (Eq. 4.29):
    dk = jtwist*q grid steps for ky index q (sign of jtwist = sign of shat).  Returns a list of
    (q, [compact kx rows i_0, i_1, ...]) with kx integers p_n = p_0 + n*jtwist*q, p_0 the member with no
    predecessor inside the dealiased set; ky = 0 modes are chains of length 1."""
    kxi = [int(v) for v in O.kx_index(Nx)]
    K = (len(kxi) - 1) // 2
    row = {p: i for i, p in enumerate(kxi)}
    chains = []
    for q in range(len(O.ky_index(Ny))):
        step = jtwist * q
        for p in range(-K, K + 1):
            if step == 0:
                chains.append((q, [row[p]]))
                continue
            if abs(p - step) <= K:          # has a predecessor: not a chain start
                continue
            members, pp = [], p
            while abs(pp) <= K:
                members.append(row[pp])
                pp += step
            chains.append((q, members))
    return chains


def apply_z_operator(f, kind, gradpar, Nx, Ny, boundary="periodic", jtwist=None):
    """gradpar * d/dz (kind="d") or |gradpar| * |k_z| (kind="a") of f[z][kx][ky] (reading L2)."""
    Nz = f.shape[0]
    if boundary == "periodic":
        M = gradpar * dz_matrix(Nz) if kind == "d" else abs(gradpar) * abs_kz_matrix(Nz)
        return np.tensordot(M, f, axes=(1, 0))
    out = np.zeros_like(f, dtype=np.complex128)
    cache = {}
    for q, rows in twist_shift_chains(Nx, Ny, jtwist):
        L = len(rows)
        if L not in cache:
            cache[L] = ext_operator_matrices(Nz, L)
        M = gradpar * cache[L][0] if kind == "d" else abs(gradpar) * cache[L][1]
        # ballooning order: mode n holds theta = z - 2 pi n, so increasing theta runs through n = L-1, ..., 0
        ext = np.concatenate([f[:, rows[n], q] for n in range(L - 1, -1, -1)])
        res = M @ ext
        for n in range(L):
            out[:, rows[n], q] = res[(L - 1 - n) * Nz:(L - n) * Nz]
    return out


# ============================================================================ pieces
def jflr_all(b, Nl):
    """J_l(b) for l = -1..Nl as a dict (zero outside 0 <= l < Nl: P:205)."""
    J = {l: O.jflr(l, b) for l in range(Nl)}
    J[-1] = np.zeros_like(b)
    J[-2] = np.zeros_like(b)
    J[Nl] = np.zeros_like(b)
    return J


def h_from_g(Gs, Phi, Jl, zt):
    """H_{l,m} = G_{l,m} + (Z/tau) J_l Phi delta_{m0}  (Eq. 4.8) for one species: [m][l][z][kx][ky]."""
    H = np.array(Gs, dtype=np.complex128, copy=True)
    for l in range(H.shape[1]):
        H[0, l] += zt * Jl[l] * Phi
    return H


def drift_frequencies(kx, ky, geo, shat):
    """(w_d^kappa, w_d^gradB)[z][kx][ky]  (reading L3)."""
    kx = np.asarray(kx)[None, :, None]
    ky = np.asarray(ky)[None, None, :]
    g = lambda n: np.asarray(geo[n], np.float64)[:, None, None]
    wk = 0.5 * (ky * g("cvdrift") + kx * g("cvdrift0") / shat)
    wb = 0.5 * (ky * g("gbdrift") + kx * g("gbdrift0") / shat)
    return wk, wb


def jtwist_of(dkx, dky, shat):
    """Signed number of kx grid steps per ky step in the twist-and-shift condition: 2 pi shat dky / dkx."""
    j = 2.0 * math.pi * shat * dky / dkx
    if abs(j - round(j)) > 1e-6 or round(j) == 0:
        raise ValueError("box is not twist-shift quantised: 2 pi shat dky/dkx = %r" % j)
    return int(round(j))


def end_damping_profile(Nz, Nx, Ny, A, width_frac=0.125, boundary="periodic", jtwist=None):
    """d[z][kx][ky] of the wave-absorbing layer, Eq. 4.30: d(zh) = A [1 - 2 zh^2/(1 + zh^4)] for
    |zh| < 1, zh = (theta - theta_end)/z_width the distance from either end of the extended z domain in units
    of z_width = width_frac * L_z (L_z/8), L_z = 2 pi L the length of the extended domain of L linked
    modes; zero elsewhere and for the zonal modes ky = 0.  Mode n of a chain holds theta = z - 2 pi n (reading L2),
    so the domain runs from theta_lo = -pi - 2 pi (L-1) to theta_hi = pi; boundary="periodic": every mode is
    its own domain (L = 1).  The end theta_hi itself is not a grid point (periodic grid z_i = -pi + 2 pi i/Nz)."""
    nakx, naky = O.dealiased_counts(Nx, Ny)
    z = -math.pi + 2.0 * math.pi * np.arange(Nz) / Nz
    d = np.zeros((Nz, nakx, naky))
    if boundary == "periodic":
        chains = [(q, [i]) for q in range(naky) for i in range(nakx)]
    else:
        chains = twist_shift_chains(Nx, Ny, jtwist)
    for q, rows in chains:
        if q == 0:
            continue
        L = len(rows)
        Lz = 2.0 * math.pi * L
        w = width_frac * Lz
        th_lo, th_hi = -math.pi - 2.0 * math.pi * (L - 1), math.pi
        for n, i in enumerate(rows):
            theta = z - 2.0 * math.pi * n
            for dist in (theta - th_lo, th_hi - theta):
                zh = dist / w
                inside = zh < 1.0
                d[inside, i, q] += A * (1.0 - 2.0 * zh[inside] ** 2 / (1.0 + zh[inside] ** 4))
    return d


def linear_rhs(G, Phi, Nx, Ny, dkx, dky, shat, geo, species, D_hyper=0.05, n_hyper=4, f_hyp=1.0,
               terms=("stream", "mirror", "drift", "drive", "coll", "hypervisc", "hypercoll"),
               boundary="periodic", damping=None):
    """dG/dt from every term of Eq. 4.9 except the nonlinear one (see module header).  fp64.
    G [s][m][l][z][kx][ky], Phi [z][kx][ky]; geo holds the per-z arrays of P:677-694 plus gradpar.
    ``terms`` selects contributions (the pins test them one at a time)."""
    G = np.asarray(G).astype(np.complex128)
    Phi = np.asarray(Phi).astype(np.complex128)
    Ns, Nm, Nl, Nz, nakx, naky = G.shape
    kx, ky = dkx * O.kx_index(Nx), dky * O.ky_index(Ny)
    kp2 = O.kperp2(kx, ky, geo["gds2"], geo["gds21"], geo["gds22"], shat)
    gradpar = float(geo["gradpar"])
    jtw = jtwist_of(dkx, dky, shat) if boundary == "linked" else None
    bgrad = np.asarray(geo["bgrad"], np.float64)[:, None, None]    # grad_par ln B
    wk, wb = drift_frequencies(kx, ky, geo, shat)
    iky = 1j * ky[None, None, :]
    kp2max = float(np.max(kp2))
    out = np.zeros_like(G)
    dend = None
    if damping is not None and damping.get("A", 0.0) != 0.0:                           # Eq. 4.30 (optional)
        dend = end_damping_profile(Nz, Nx, Ny, damping["A"], damping.get("width_frac", 0.125), boundary, jtw)
    dpar = lambda f: apply_z_operator(f, "d", gradpar, Nx, Ny, boundary, jtw)          # grad_par
    kpar = lambda f: apply_z_operator(f, "a", gradpar, Nx, Ny, boundary, jtw)          # |k_par|
    for s, sp in enumerate(species):
        Z, mass, temp = _get(sp, "Z"), _get(sp, "mass"), _get(sp, "temp")
        tprim, fprim, nu = _get(sp, "tprim"), _get(sp, "fprim"), _nu(sp)
        vt = math.sqrt(temp / mass)
        zt, tz = Z / temp, temp / Z
        b = O.b_species(kp2, geo["bmag"], Z, mass, temp)
        J = jflr_all(b, Nl)
        H = h_from_g(G[s], Phi, J, zt)

        def Hlm(l, m):
            if 0 <= l < Nl and 0 <= m < Nm:
                return H[m, l]
            return 0.0

        # field-particle moments of the Dougherty operator, Eq. 4.14-4.18
        upar = sum(J[l] * Hlm(l, 1) for l in range(Nl))
        uperp = np.sqrt(b) * sum((J[l] + J[l - 1]) * Hlm(l, 0) for l in range(Nl))
        Tpar = math.sqrt(2.0) * sum(J[l] * Hlm(l, 2) for l in range(Nl))
        Tperp = sum((l * J[l - 1] + 2 * l * J[l] + (l + 1) * J[l + 1]) * Hlm(l, 0) for l in range(Nl))
        Tbar = (Tpar + 2.0 * Tperp) / 3.0
        p_hyp = Nm / 2.0
        m_max = max(Nm - 1, 1)
        nuhyp_fac = 2.5 * f_hyp * (p_hyp + 0.5) / m_max ** (p_hyp + 0.5) * vt

        for m in range(Nm):
            for l in range(Nl):
                r = np.zeros((Nz, nakx, naky), dtype=np.complex128)
                if "stream" in terms:
                    r -= vt * dpar(math.sqrt(m + 1) * Hlm(l, m + 1) + math.sqrt(m) * Hlm(l, m - 1)
                                   + np.zeros((Nz, nakx, naky)))
                if "mirror" in terms:
                    r -= vt * bgrad * (-(l + 1) * math.sqrt(m + 1) * Hlm(l, m + 1)
                                       - l * math.sqrt(m + 1) * Hlm(l - 1, m + 1)
                                       + l * math.sqrt(m) * Hlm(l, m - 1)
                                       + (l + 1) * math.sqrt(m) * Hlm(l + 1, m - 1))
                if "drift" in terms:
                    r -= 1j * tz * wk * (math.sqrt((m + 1) * (m + 2)) * Hlm(l, m + 2) + (2 * m + 1) * Hlm(l, m)
                                         + math.sqrt(m * (m - 1)) * Hlm(l, m - 2))
                    r -= 1j * tz * wb * ((l + 1) * Hlm(l + 1, m) + (2 * l + 1) * Hlm(l, m) + l * Hlm(l - 1, m))
                if "drive" in terms:
                    if m == 0:
                        r += iky * (fprim * J[l] + tprim * (l * J[l - 1] + 2 * l * J[l] + (l + 1) * J[l + 1])) * Phi
                    elif m == 2:
                        r += iky * tprim * J[l] * Phi / math.sqrt(2.0)
                if "coll" in terms and nu != 0.0:
                    r -= nu * (b + 2 * l + m) * Hlm(l, m)
                    if m == 0:
                        r += nu * (np.sqrt(b) * (J[l] + J[l - 1]) * uperp
                                   + 2.0 * (l * J[l - 1] + 2 * l * J[l] + (l + 1) * J[l + 1]) * Tbar)
                    elif m == 1:
                        r += nu * J[l] * upar
                    elif m == 2:
                        r += nu * math.sqrt(2.0) * J[l] * Tbar
                if "hypervisc" in terms and D_hyper != 0.0:
                    r -= D_hyper * (kp2 / kp2max) ** n_hyper * G[s, m, l]
                if "hypercoll" in terms and f_hyp != 0.0 and m > 2:
                    r -= nuhyp_fac * float(m) ** p_hyp * kpar(G[s, m, l])
                if dend is not None:
                    r -= dend * Hlm(l, m)                                   # Eq. 4.30: acts on H, ky != 0 only
                out[s, m, l] = r
    return out


# ============================================================================ full RHS and time step
def rhs(G, Nx, Ny, dkx, dky, shat, geo, species, tau_fac=1.0, adiabatic=None, D_hyper=0.05, n_hyper=4,
        f_hyp=1.0, nonlinear=True, planes=None, boundary="periodic", damping=None):
    """gx_rhs: Phi from quasineutrality, then -N + linear terms (Eq. 4.9)."""
    adiabatic = (len(species) == 1) if adiabatic is None else adiabatic
    Phi = O.field_solve(G, Nx, Ny, dkx, dky, shat, geo, species, tau_fac=tau_fac, adiabatic=adiabatic)
    out = linear_rhs(G, Phi, Nx, Ny, dkx, dky, shat, geo, species, D_hyper, n_hyper, f_hyp, boundary=boundary,
                     damping=damping)
    if nonlinear:
        out = out + O.nonlinear_rhs(G, Phi, Nx, Ny, dkx, dky, shat, geo, species, method="dft", planes=planes)
    return out


def ssp_rk3_step(y, dt, f):
    """Third-order strong-stability-preserving Runge-Kutta, Shu-Osher form (reading L8):
    y1 = y + dt f(y);  y2 = 3/4 y + 1/4 (y1 + dt f(y1));  y_new = 1/3 y + 2/3 (y2 + dt f(y2))."""
    y1 = y + dt * f(y)
    y2 = 0.75 * y + 0.25 * (y1 + dt * f(y1))
    return y / 3.0 + 2.0 / 3.0 * (y2 + dt * f(y2))
