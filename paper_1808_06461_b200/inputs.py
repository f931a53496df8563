"""Seeded synthetic inputs shared by the oracle-side tests and the CUDA-side tests / bench.

Holds NONE of the method's arithmetic (no compact differences, no banded solves, no dealiased
products): fields are analytic polynomials in y times random Fourier amplitudes, so every derivative
used here is an exact polynomial derivative.  Recipe: for every retained
(p,q) != (0,0)

    v^(y)    = a(k) (1-y^2)^2 sum_{m<M} c_m T_m(y)/(m+1)       (v = dv/dy = 0 at the walls)
    om_y^(y) = a(k) (1-y^2)   sum_{m<M} d_m T_m(y)/(m+1)       (om_y = 0 at the walls)
    phi^     = v^'' - k^2 v^                                    (analytic)

c_m, d_m complex standard normal from one seeded generator; the p = 0 column is made Hermitian in q;
one global rescale.  These stand in for the paper's turbulent fields (Table 2.1,
Table 3.1; the production initial data of L159 are not available).
"""
import math

import numpy as np
import torch
from numpy.polynomial import chebyshev as _cheb
from numpy.polynomial import polynomial as _poly


# ---------------------------------------------------------------------------------- meshes (R10)
def mesh_cosine(ny, a=0.7):
    xi = np.linspace(-1.0, 1.0, ny)
    y = np.sin(a * np.pi * xi / 2.0) / math.sin(a * np.pi / 2.0)
    return _symmetrise(y)


def mesh_tanh(ny, gamma):
    xi = np.linspace(-1.0, 1.0, ny)
    y = np.tanh(gamma * xi) / math.tanh(gamma)
    return _symmetrise(y)


def _symmetrise(y):
    y = 0.5 * (y - y[::-1])
    y[0], y[-1] = -1.0, 1.0
    if y.size % 2:
        y[y.size // 2] = 0.0
    return y


# ---------------------------------------------------------------------------------- mean profiles
def mean_poiseuille(y, ucl):
    return ucl * (1.0 - y * y)


def mean_reichardt(y, re_tau, kappa=0.41):
    yp = re_tau * (1.0 - np.abs(y))
    return np.log1p(kappa * yp) / kappa + 7.8 * (1.0 - np.exp(-yp / 11.0) - (yp / 11.0) * np.exp(-yp / 3.0))


# ---------------------------------------------------------------------------------- configs
CONFIGS = {
    # name: grid, box, nu^-1, dt, mesh, mean, spectrum, M, filter cutoffs
    "cfg1": dict(nx=32, ny=33, nz=32, lx=2 * math.pi, lz=math.pi, re=180.0, dt=1e-3, mesh=("cos", 0.7),
                 mean=("poiseuille", 90.0), spec="gauss", M=6, amp=("maxu", 1e-3 * 90.0), cut=(8, 8), seed=1),
    "cfg2": dict(nx=16, ny=129, nz=4, lx=2 * math.pi, lz=2 * math.pi / 3, re=7500.0, dt=5e-3, mesh=("tanh", 2.5),
                 mean=("poiseuille", 1.0), spec=None, M=0, amp=None, cut=(1, 1), seed=2),
    "cfg3": dict(nx=768, ny=251, nz=576, lx=8 * math.pi, lz=3 * math.pi, re=550.0, dt=2e-4, mesh=("tanh", 2.5),
                 mean=("reichardt", 550.0), spec="vk", M=8, amp=("rms", 1.0), cut=(95, 71), seed=3),
    "cfg4": dict(nx=1024, ny=633, nz=1024, lx=2 * math.pi, lz=math.pi, re=2000.0, dt=4e-5, mesh=("tanh", 2.72),
                 mean=("reichardt", 2000.0), spec="vk", M=8, amp=("rms", 1.0), cut=(62, 62), seed=4),
    "cfg5": dict(nx=1536, ny=1025, nz=1152, lx=0.8 * math.pi, lz=0.3 * math.pi, re=5300.0, dt=1e-5,
                 mesh=("tanh", 3.0), mean=("reichardt", 5300.0), spec="vk", M=8, amp=("rms", 1.0), cut=(95, 71), seed=5),
    # config 5 on a 129-plane slab: the same planes, transform plans, tiles and chunks as cfg5 in 1/8 of the memory
    # (ncu --set full backs the device memory up on the host, which the 146 GB workspace of cfg5 does not survive)
    "cfg5slab": dict(nx=1536, ny=129, nz=1152, lx=0.8 * math.pi, lz=0.3 * math.pi, re=5300.0, dt=1e-5,
                     mesh=("tanh", 2.5), mean=("reichardt", 5300.0), spec="vk", M=8, amp=("rms", 1.0), cut=(95, 71), seed=5),
    # mid-size parity case: several FFT/solver tiles plus ragged tails, oracle finishes in seconds
    "mid": dict(nx=96, ny=65, nz=48, lx=4 * math.pi, lz=2 * math.pi, re=180.0, dt=5e-4, mesh=("cos", 0.8),
                mean=("reichardt", 180.0), spec="vk", M=8, amp=("rms", 1.0), cut=(11, 7), seed=7),
}


def config(name, **over):
    c = dict(CONFIGS[name])
    c.update(over)
    kind, par = c["mesh"]
    c["y"] = mesh_cosine(c["ny"], par) if kind == "cos" else mesh_tanh(c["ny"], par)
    mk, mp = c["mean"]
    c["U"] = mean_poiseuille(c["y"], mp) if mk == "poiseuille" else mean_reichardt(c["y"], mp)
    c["W"] = np.zeros(c["ny"])
    return c


# ---------------------------------------------------------------------------------- fluctuations
def _basis_tables(y, M):
    """P_m = (1-y^2)^2 T_m/(m+1), its first two y-derivatives, and Q_m = (1-y^2) T_m/(m+1) on the mesh."""
    P = np.zeros((3, M, y.size))
    Q = np.zeros((M, y.size))
    w2 = _poly.polypow([1.0, 0.0, -1.0], 2)
    w1 = np.array([1.0, 0.0, -1.0])
    for m in range(M):
        t = _cheb.cheb2poly([0.0] * m + [1.0]) / (m + 1.0)
        p = _poly.polymul(w2, t)
        P[0, m] = _poly.polyval(y, p)
        P[1, m] = _poly.polyval(y, _poly.polyder(p, 1))
        P[2, m] = _poly.polyval(y, _poly.polyder(p, 2))
        Q[m] = _poly.polyval(y, _poly.polymul(w1, t))
    return P, Q


def _amplitude(k2, spec):
    if spec == "gauss":  # energy ~ exp(-(kx^2+kz^2)/8)
        return torch.exp(-k2 / 16.0)
    kh = torch.sqrt(k2) / 4.0  # von Karman-like E(k) ~ k^4/(1+k^2)^(17/6)
    e = kh ** 4 / (1.0 + kh * kh) ** (17.0 / 6.0)
    return torch.sqrt(e / torch.clamp(kh, min=1e-30))


def fluctuations(c, device="cpu", layout="line", zchunk=None, out=None):
    """Seeded (v^, phi^, om_y^) for config dict ``c``; complex128 torch tensors on ``device``.

    layout "line": [nz][nx/2][ny] (the C ABI's state layout).  The rescale uses only analytic
    quantities (u^, w^ from the polynomial dv/dy): "maxu" = max over the nx x nz collocation grid of
    |u - <u>|, "rms" = plane- and y-point-averaged (u'^2+v'^2+w'^2)/3 = amp^2.
    ``zchunk``: build the fields in slabs of that many k_z slots (bounds the temporaries for the large
    configs; "rms" rescale only).  ``out``: optional triple of preallocated [nz][nx/2][ny] complex128
    tensors (any device, e.g. pinned host memory) that receive the result slab by slab.
    """
    nx, ny, nz, M = c["nx"], c["ny"], c["nz"], c["M"]
    nxh, nzh = nx // 2, nz // 2
    dev = torch.device(device)
    g = torch.Generator(device="cpu").manual_seed(int(c["seed"]))
    coef = torch.randn((2, nz, nxh, M, 2), generator=g, dtype=torch.float64)
    coef = torch.view_as_complex(coef).to(dev)  # [2][nz][nxh][M]
    # Hermitian p = 0 column: f(0,-q) = conj f(0,q)
    for q in range(1, nzh):
        coef[:, nz - q, 0, :] = torch.conj(coef[:, q, 0, :])
    coef[:, nzh, :, :] = 0.0
    coef[:, 0, 0, :] = 0.0
    kx = 2.0 * math.pi * torch.arange(nxh, dtype=torch.float64, device=dev) / c["lx"]
    qs = torch.cat([torch.arange(nzh), torch.zeros(1, dtype=torch.long), torch.arange(-nzh + 1, 0)]).to(dev)
    kz = 2.0 * math.pi * qs.to(torch.float64) / c["lz"]
    k2 = kz[:, None] ** 2 + kx[None, :] ** 2
    amp = _amplitude(k2, c["spec"])
    amp[0, 0] = 0.0
    amp[nzh, :] = 0.0
    P, Q = _basis_tables(c["y"], M)
    P = torch.from_numpy(P).to(dev).to(torch.complex128)
    Q = torch.from_numpy(Q).to(dev).to(torch.complex128)
    k2s = k2.clone()
    k2s[0, 0] = 1.0
    k2s[nzh, :] = 1.0
    kind, target = c["amp"]
    step = nz if (zchunk is None or kind == "maxu") else int(zchunk)
    if out is None:
        out = tuple(torch.empty((nz, nxh, ny), dtype=torch.complex128, device=dev) for _ in range(3))
    wp = torch.full((nxh,), 2.0, dtype=torch.float64, device=dev)
    wp[0] = 1.0
    def slab(sl):
        cv = coef[0, sl] * amp[sl, :, None]
        cw = coef[1, sl] * amp[sl, :, None]
        v = cv @ P[0]
        dv = cv @ P[1]
        phi = cv @ P[2] - k2[sl, :, None] * v
        omy = cw @ Q
        return v, dv, phi, omy

    slabs = [slice(z0, min(nz, z0 + step)) for z0 in range(0, nz, step)]
    esum, umax, keep = 0.0, 0.0, None
    for sl in slabs:  # pass 1: the norm used by the rescale (analytic u^, w^)
        v, dv, phi, omy = slab(sl)
        u = 1j * (kx[None, :, None] * dv - kz[sl, None, None] * omy) / k2s[sl, :, None]
        w = 1j * (kz[sl, None, None] * dv + kx[None, :, None] * omy) / k2s[sl, :, None]
        del dv
        if kind == "maxu":
            full = torch.zeros((nz, nxh + 1, ny), dtype=torch.complex128, device=dev)
            full[:, :nxh] = u
            phys = torch.fft.irfft(torch.fft.ifft(full, dim=0) * nz, n=nx, dim=1) * nx
            umax = float(phys.abs().max())
        else:
            esum += float(((u.abs() ** 2 + v.abs() ** 2 + w.abs() ** 2) * wp[None, :, None]).sum())
        del u, w
        keep = (v, phi, omy) if len(slabs) == 1 else None
    scale = target / umax if kind == "maxu" else target / math.sqrt(esum / (3.0 * ny))
    for sl in slabs:  # pass 2: rescaled fields, slab by slab
        v, phi, omy = keep if keep is not None else [t for n, t in enumerate(slab(sl)) if n != 1]
        out[0][sl].copy_(v * scale)
        out[1][sl].copy_(phi * scale)
        out[2][sl].copy_(omy * scale)
        del v, phi, omy
    keep = None
    v, phi, omy = out
    if layout == "plane":
        v, phi, omy = (t.permute(2, 0, 1).contiguous() for t in (v, phi, omy))
    return v, phi, omy
