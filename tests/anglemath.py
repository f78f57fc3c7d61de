"""Angle-form lattice helpers used only by the tests (numpy, np.roll on the coordinate grid).

A second, structurally different route to the same quantities the oracle computes with complex
arithmetic and neighbour tables: F = sum cos(theta^g), Delta_i = sum_mu [sin theta^g_{i,mu} - sin theta^g_{i-mu,mu}],
theta^g_{i,mu} = theta_{i,mu} + phi_i - phi_{i+mu}  (Eq. 3 PAPER.md:L58 in the Eq. 5 convention, L38).
Arrays are shaped with x0 fastest: theta.reshape(N_{d-1},...,N_0,d), phi.reshape(N_{d-1},...,N_0);
direction mu lives on numpy axis d-1-mu.
"""
import itertools

import numpy as np


def shape(ext):
    return tuple(int(n) for n in ext[::-1])


def axis(ext, mu):
    return len(ext) - 1 - mu


def gauged_angles(ext, theta, phi):
    d = len(ext)
    th = np.asarray(theta, dtype=np.float64).reshape(shape(ext) + (d,))
    ph = np.asarray(phi, dtype=np.float64).reshape(shape(ext))
    out = np.empty_like(th)
    for mu in range(d):
        out[..., mu] = th[..., mu] + ph - np.roll(ph, -1, axis=axis(ext, mu))
    return out


def functional(ext, theta, phi):
    return float(np.cos(gauged_angles(ext, theta, phi)).sum())


def divergence(ext, theta, phi):
    tg = gauged_angles(ext, theta, phi)
    D = np.zeros(shape(ext))
    for mu in range(len(ext)):
        s = np.sin(tg[..., mu])
        D += s - np.roll(s, 1, axis=axis(ext, mu))
    return D.reshape(-1)


def fp_matrix(ext, theta, phi):
    """M = Hessian of -F w.r.t. phi: cos-weighted Laplacian."""
    d = len(ext)
    V = int(np.prod(ext))
    c = np.cos(gauged_angles(ext, theta, phi))
    idx = np.arange(V).reshape(shape(ext))
    M = np.zeros((V, V))
    for mu in range(d):
        j = np.roll(idx, -1, axis=axis(ext, mu)).reshape(-1)
        i = idx.reshape(-1)
        cm = c[..., mu].reshape(-1)
        np.add.at(M, (i, i), cm)
        np.add.at(M, (j, j), cm)
        np.add.at(M, (i, j), -cm)
        np.add.at(M, (j, i), -cm)
    return M


def plaquettes(ext, theta):
    """theta_{i,mu} + theta_{i+mu,nu} - theta_{i+nu,mu} - theta_{i,nu} for mu<nu, wrapped to (-pi,pi]."""
    d = len(ext)
    th = np.asarray(theta, dtype=np.float64).reshape(shape(ext) + (d,))
    out = []
    for mu, nu in itertools.combinations(range(d), 2):
        p = (th[..., mu] + np.roll(th[..., nu], -1, axis=axis(ext, mu))
             - np.roll(th[..., mu], -1, axis=axis(ext, nu)) - th[..., nu])
        out.append(np.angle(np.exp(1j * p)).reshape(-1))
    return np.array(out)


def to_g(phi):
    phi = np.asarray(phi, dtype=np.float64).reshape(-1)
    return np.stack([np.cos(phi), np.sin(phi)], axis=1)


def to_phi(g):
    g = np.asarray(g).reshape(-1, 2)
    return np.arctan2(g[:, 1], g[:, 0])


def coords(ext):
    """x[i, mu] for site index i (x0 fastest)."""
    V = int(np.prod(ext))
    i = np.arange(V)
    x = np.zeros((V, len(ext)), dtype=np.int64)
    for mu, n in enumerate(ext):
        x[:, mu] = i % n
        i = i // n
    return x


def phased_sweep(ext, theta, g, omega, naive_two_colour=False):
    """Concurrent (Jacobi-within-phase) sweep: parity p = 0,1; inside a parity class the phases are the levels
    l(i) = #{mu : N_mu odd and x_mu = N_mu - 1} (reading R3).  With naive_two_colour the level split
    is dropped (wrong on odd extents; used to show the readings differ)."""
    d = len(ext)
    x = coords(ext)
    par = x.sum(1) % 2
    lvl = np.zeros(len(x), dtype=np.int64)
    for mu, n in enumerate(ext):
        if n % 2 == 1:
            lvl += (x[:, mu] == n - 1)
    if naive_two_colour:
        lvl[:] = 0
    V = len(x)
    idx = np.arange(V).reshape(shape(ext))
    fwd = [np.roll(idx, -1, axis=axis(ext, mu)).reshape(-1) for mu in range(d)]
    bwd = [np.roll(idx, 1, axis=axis(ext, mu)).reshape(-1) for mu in range(d)]
    U = np.exp(1j * np.asarray(theta).reshape(V, d))
    gc = np.asarray(g)[:, 0] + 1j * np.asarray(g)[:, 1]
    for p in (0, 1):
        for l in range(lvl.max() + 1):
            s = np.nonzero((par == p) & (lvl == l))[0]
            if not len(s):
                continue
            w = np.zeros(len(s), dtype=complex)
            for mu in range(d):
                w += np.conj(U[s, mu]) * gc[fwd[mu][s]] + U[bwd[mu][s], mu] * gc[bwd[mu][s]]
            gh = w / np.abs(w)
            h = (1 - omega) * gc[s] + omega * gh
            gc[s] = h / np.abs(h)
    return np.stack([gc.real, gc.imag], axis=1)
