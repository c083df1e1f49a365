"""Exact Boltzmann sums on tiny periodic lattices, by brute-force enumeration in numpy.

Independent of oracle/ and of the CUDA path: nothing here is imported by either.  Used to pin
the oracle's stationary law (SURVEY.md section 8(c) "Pins": 4x4 enumeration, 2x2 histogram).

Conventions (Eq. 1, J = 1): H = -sum_<xy> s_x s_y + Delta * sum_x s_x^2 where
the bond sum runs over every site's right and down neighbour with periodic wrap (so on a 2x2
lattice every bond is counted twice, exactly as a site's four-neighbour sum sees it).
"""
from __future__ import annotations

import numpy as np


def _bond_sum(s: np.ndarray) -> np.ndarray:
    """s: (..., L, L) array of spins -> sum over sites of s*(right + down), periodic."""
    return (s * np.roll(s, -1, axis=-1)).sum(axis=(-1, -2)) + \
           (s * np.roll(s, -1, axis=-2)).sum(axis=(-1, -2))


def enumerate_states(L: int, values) -> np.ndarray:
    """All len(values)**(L*L) configurations as an (n, L, L) int8 array.

    State k has site x = i*L + j equal to values[digit x of k in base len(values)]."""
    q = len(values)
    n = q ** (L * L)
    k = np.arange(n, dtype=np.int64)
    out = np.empty((n, L * L), dtype=np.int8)
    vals = np.asarray(values, dtype=np.int8)
    for x in range(L * L):
        out[:, x] = vals[k % q]
        k //= q
    return out.reshape(n, L, L)


def ising_exact(L: int, beta: float) -> dict:
    s = enumerate_states(L, (-1, +1)).astype(np.int64)
    B = _bond_sum(s)
    M = s.sum(axis=(-1, -2))
    w = np.exp(beta * (B - B.max()))
    Z = w.sum()
    n = L * L
    return {
        "e": float((-(B / n) * w).sum() / Z),
        "abs_m": float((np.abs(M) / n * w).sum() / Z),
        "m2": float(((M / n) ** 2 * w).sum() / Z),
        "prob": w / Z,            # Boltzmann weight of state k (digit x = (s_x+1)/2 in base 2)
        "B": B, "M": M,
    }


def blume_capel_exact_4x4(beta: float, delta: float) -> dict:
    """<H>/N, bond part, <|m|>, <q>, <m^2> over the 3^16 states of the 4x4 lattice.

    Decomposed row by row (81 states per row) so that no array is larger than 81^3."""
    L = 4
    rows = enumerate_states(1, (-1, 0, +1)).reshape(3, 1)          # placeholder to keep API tidy
    del rows
    # all 81 rows
    k = np.arange(81)
    r = np.empty((81, 4), dtype=np.int64)
    kk = k.copy()
    for x in range(4):
        r[:, x] = kk % 3 - 1
        kk //= 3
    horiz = (r * np.roll(r, -1, axis=1)).sum(axis=1)                # bonds inside a row
    vert = r @ r.T                                                   # bonds between two rows
    m_row = r.sum(axis=1)
    q_row = (r * r).sum(axis=1)
    n = L * L
    acc = np.zeros(6)           # Z, sum H w, sum B w, sum |M| w, sum Q w, sum M^2 w
    # shift energies by the ground state so exp() stays finite
    e_shift = -2.0 * n + min(delta, 0.0) * n
    a, b, c = np.meshgrid(k, k, k, indexing="ij")                   # rows 1..3
    Bin = horiz[a] + horiz[b] + horiz[c] + vert[a, b] + vert[b, c]
    Min = m_row[a] + m_row[b] + m_row[c]
    Qin = q_row[a] + q_row[b] + q_row[c]
    for r0 in range(81):
        B = Bin + horiz[r0] + vert[r0, a] + vert[c, r0]
        M = Min + m_row[r0]
        Q = Qin + q_row[r0]
        H = -B + delta * Q
        w = np.exp(-beta * (H - e_shift))
        acc += [w.sum(), (H * w).sum(), (B * w).sum(), (np.abs(M) * w).sum(), (Q * w).sum(),
                (M.astype(np.float64) ** 2 * w).sum()]
    Z = acc[0]
    return {
        "h": acc[1] / Z / n,
        "bond": -acc[2] / Z / n,
        "abs_m": acc[3] / Z / n,
        "q": acc[4] / Z / n,
        "m2": acc[5] / Z / n / n,
    }


def small_exact(L: int, values, beta: float, delta: float = 0.0) -> dict:
    """Boltzmann probabilities of every state of a tiny lattice (2x2), base-len(values) codes."""
    s = enumerate_states(L, values).astype(np.int64)
    B = _bond_sum(s)
    Q = (s * s).sum(axis=(-1, -2))
    H = -B + delta * Q
    w = np.exp(-beta * (H - H.min()))
    return {"prob": w / w.sum(), "states": s}


def sweep_matrix(L: int, values, beta: float, delta: float = 0.0) -> np.ndarray:
    """Exact transition matrix of one checkerboard Metropolis sweep (black then white) on a
    tiny periodic lattice, built from the definition: within a half-sweep the sites of one
    colour are updated independently; Ising proposes the flip, Blume-Capel one of the two
    other values with probability 1/2 each; acceptance min(1, exp(-beta*dE)), dE from Eq. (1).
    State codes as in `enumerate_states`."""
    q = len(values)
    n = L * L
    states = enumerate_states(L, values).astype(np.int64).reshape(-1, n)
    ns = states.shape[0]
    code = {tuple(s): k for k, s in enumerate(states)}
    P = np.eye(ns)
    for colour in (0, 1):
        H = np.zeros((ns, ns))
        sites = [(i, j) for i in range(L) for j in range(L) if (i + j) % 2 == colour]
        for k, s in enumerate(states):
            g = s.reshape(L, L)
            dist = {tuple(s): 1.0}
            for (i, j) in sites:
                h = g[(i - 1) % L, j] + g[(i + 1) % L, j] + g[i, (j - 1) % L] + g[i, (j + 1) % L]
                cur = g[i, j]
                others = [v for v in values if v != cur]
                move = {}
                for v in others:
                    dE = -(v - cur) * h + delta * (v * v - cur * cur)
                    move[v] = min(1.0, np.exp(-beta * dE)) / len(others)
                stay = 1.0 - sum(move.values())
                new = {}
                for st, pr in dist.items():
                    for v, pv in list(move.items()) + [(cur, stay)]:
                        t = list(st)
                        t[i * L + j] = v
                        new[tuple(t)] = new.get(tuple(t), 0.0) + pr * pv
                dist = new
            for st, pr in dist.items():
                H[k, code[st]] += pr
        P = P @ H
    return P


def cesaro_limit(P: np.ndarray, start: int, doublings: int = 24) -> np.ndarray:
    """lim (1/n) sum_{k<n} e_start P^k, by repeated doubling (handles periodic/reducible chains)."""
    A = np.eye(P.shape[0])
    Pn = P.copy()
    for _ in range(doublings):
        A = 0.5 * (A + Pn @ A)
        Pn = Pn @ Pn
    return A[start]


def binned_error(x: np.ndarray, nbins: int = 50):
    """Mean and standard error from bin averages (handles autocorrelation)."""
    x = np.asarray(x, dtype=np.float64)
    n = (x.size // nbins) * nbins
    bins = x[:n].reshape(nbins, -1).mean(axis=1)
    return float(bins.mean()), float(bins.std(ddof=1) / np.sqrt(nbins))
