"""Estimator layer: from many independent runs to xi(t) and z.

Host-side fp64 analysis of the integer counts the CUDA path returns; nothing here touches the
device.  It restates the procedures of the paper:

* errors by the jackknife over independent realisations (App. C, D);
* the coherence length xi = I_2 / I_1, I_n = int_0^inf r^n C(r) dr (Eq. C1) with
  the paper's three steps: (i) r_cut where C(r_cut + 1) drops below three
  times its error; (ii) r* = argmax r^2 C, r_min / r_max the first r where r^2 C falls below
  0.9 / (1/3) of that maximum; (iii) if r_max - r_min <= 8 integrate the data up to r_cut, else
  fit F(r) = A exp[-(r/xi_F)^beta] / sqrt(r) (Eq. C2) on [r_min, r_max], integrate the data up
  to r_max and F from r_max to 20 xi_F.  Our C(r) is dense in r (reading 9), so the
  paper's cubic-spline interpolation of a sparse r-grid is not needed;
* the dynamic exponent z from log t = z log xi + b + b' xi^(-omega), omega = 1.75 (Eq. 5 / D1,
  PAPER.md:75-81, 223-225), least squares with the error of xi propagated through the
  derivative of the fitting function, chi^2/dof and the fit quality
  Q = Gamma(dof/2, chi^2/2) / Gamma(dof/2), errors by the jackknife.
"""
from __future__ import annotations

import numpy as np

OMEGA = 1.75          # corrections-to-scaling exponent used by the paper


def jackknife(samples: np.ndarray, estimator=None):
    """samples[run, ...] -> (estimate on the mean of all runs, jackknife error).

    estimator maps the mean over a set of runs to the quantity of interest (default: identity).
    Leave-one-out means; error^2 = (N-1)/N * sum (theta_i - theta_bar)^2."""
    x = np.asarray(samples, dtype=np.float64)
    n = x.shape[0]
    if n < 2:
        raise ValueError("the jackknife needs at least two runs")
    f = (lambda a: a) if estimator is None else estimator
    total = x.sum(axis=0)
    full = np.asarray(f(total / n), dtype=np.float64)
    loo = np.array([np.asarray(f((total - x[i]) / (n - 1)), dtype=np.float64) for i in range(n)])
    err = np.sqrt((n - 1) / n * ((loo - loo.mean(axis=0)) ** 2).sum(axis=0))
    return full, err


def correlation(Sx, Sy, L: int, Q=None) -> np.ndarray:
    """C(r) for r = 0..r_max from the axis sums of one run: C(0) = Q / L^2 (1 for Ising),
    C(r) = (S_x(r) + S_y(r)) / (2 L^2) (reading 10)."""
    n = float(L) * float(L)
    c0 = 1.0 if Q is None else float(Q) / n
    return np.concatenate([[c0], (np.asarray(Sx, np.float64) + np.asarray(Sy, np.float64)) / (2.0 * n)])


def _F(r, A, xiF, beta):
    return A * np.exp(-(r / xiF) ** beta) / np.sqrt(r)


class CutoffWarning(UserWarning):
    """The ordering r* < r_min < r_max <= r_cut that App. C requires was not found."""


def xi_appendix_c(C: np.ndarray, C_err: np.ndarray, details: dict | None = None, cutoffs: dict | None = None,
                  strict: bool = False) -> float:
    """xi = I_2 / I_1 by the paper's procedure (module docstring); C[r], C_err[r] for r = 0..R.

    cutoffs = {"r_cut", "r_min", "r_max"} freezes the three cut-offs (the jackknife passes the
    full sample's, so that every leave-one-out mean is integrated over the same ranges).  The
    paper requires r* < r_min < r_max < r_cut and asks for more statistics otherwise
    (PAPER.md:202-207); when r_min or r_max is not found before r_cut this routine integrates the
    data up to r_cut only, which biases xi low: details["condition_met"] is then False and a
    CutoffWarning is issued (strict=True raises ValueError instead)."""
    import warnings
    C = np.asarray(C, np.float64)
    E = np.asarray(C_err, np.float64)
    R = C.size - 1
    r = np.arange(R + 1, dtype=np.float64)
    if cutoffs is None:
        # (i) cut-off: the last r before C(r + 1) < 3 err(r + 1)
        bad = np.nonzero(C[1:] < 3.0 * E[1:])[0]
        r_cut = int(bad[0]) if bad.size else R               # bad[0] indexes C[1:], i.e. r = bad[0] + 1
        if r_cut < 2:
            raise ValueError("the correlation function is noise from r = 2 on")
        w = r[: r_cut + 1] ** 2 * C[: r_cut + 1]
        r_star = int(np.argmax(w))
        below = lambda frac: next((int(k) for k in range(r_star + 1, r_cut + 1) if w[k] < frac * w[r_star]), None)
        r_min, r_max = below(0.9), below(1.0 / 3.0)
    else:
        r_cut, r_min, r_max = cutoffs["r_cut"], cutoffs["r_min"], cutoffs["r_max"]
        r_star = cutoffs.get("r_star")
    found = r_min is not None and r_max is not None
    info = {"r_cut": r_cut, "r_star": r_star, "r_min": r_min, "r_max": r_max, "tail_fit": False,
            "condition_met": bool(found)}
    if not found:
        msg = (f"App. C cut-offs not found before r_cut = {r_cut} (r_min = {r_min}, r_max = {r_max}): "
               "integrating the data up to r_cut only biases xi low; more statistics or a larger r range needed")
        if strict:
            raise ValueError(msg)
        warnings.warn(msg, CutoffWarning, stacklevel=2)

    def trapz(n, upto):
        y = r[: upto + 1] ** n * C[: upto + 1]
        return float(np.sum(0.5 * (y[1:] + y[:-1])))

    if not found or r_max - r_min <= 8:
        I1, I2 = trapz(1, r_cut), trapz(2, r_cut)             # (iii), first branch
    else:
        from scipy.optimize import curve_fit
        rr = r[r_min: r_max + 1]
        sig = np.maximum(E[r_min: r_max + 1], 1e-300)
        xi0 = max(float(r_star if r_star is not None else r_min), 1.0)
        p0 = (C[r_min] * np.sqrt(rr[0]) * np.e, xi0, 1.5)
        popt, _ = curve_fit(_F, rr, C[r_min: r_max + 1], p0=p0, sigma=sig, maxfev=20000,
                            bounds=([0.0, 1e-3, 0.1], [np.inf, np.inf, 10.0]))
        A, xiF, beta = (float(v) for v in popt)
        info.update(tail_fit=True, A=A, xi_F=xiF, beta=beta)
        upper = max(20.0 * xiF, float(r_max) + 1.0)
        fine = np.linspace(float(r_max), upper, 20001)

        def tail(n):
            y = fine ** n * _F(fine, A, xiF, beta)
            return float(np.sum(0.5 * (y[1:] + y[:-1]) * np.diff(fine)))

        I1, I2 = trapz(1, r_max) + tail(1), trapz(2, r_max) + tail(2)
    if details is not None:
        details.update(info, I1=I1, I2=I2)
    return I2 / I1


def xi_with_error(C_runs: np.ndarray, details: dict | None = None):
    """C_runs[run, r] -> (xi, jackknife error).  The cut-offs r_cut, r_min, r_max are fixed ONCE
    from the full sample's mean and error and reused for every leave-one-out mean;
    the tail fit itself is repeated on each of them."""
    import warnings
    C_runs = np.asarray(C_runs, np.float64)
    n = C_runs.shape[0]
    err = C_runs.std(axis=0, ddof=1) / np.sqrt(n)
    d = {}
    xi_appendix_c(C_runs.mean(axis=0), err, d)                 # warns once if the condition fails
    frozen = {k: d[k] for k in ("r_cut", "r_star", "r_min", "r_max")}
    if details is not None:
        details.update(d)
    with warnings.catch_warnings():
        warnings.simplefilter("ignore", CutoffWarning)
        xi, xi_err = jackknife(C_runs, lambda m: xi_appendix_c(m, err, cutoffs=frozen))
    return float(xi), float(xi_err)


def _fit_z_once(logt, xi, xi_err, omega):
    """Weighted linear least squares of log t = z log xi + b + b' xi^-omega; the weights use the
    error of xi propagated through f'(xi), iterated to self-consistency."""
    X = np.stack([np.log(xi), np.ones_like(xi), xi ** (-omega)], axis=1)
    sigma = np.maximum(xi_err / xi, 1e-300)                       # start: f' ~ z / xi with z ~ 1
    for _ in range(20):
        W = 1.0 / sigma
        p, *_ = np.linalg.lstsq(X * W[:, None], logt * W, rcond=None)
        fprime = p[0] / xi - omega * p[2] * xi ** (-omega - 1.0)
        new = np.maximum(1e-40 + xi_err * np.abs(fprime), 1e-300)  # t_error = 1e-40
        if np.allclose(new, sigma, rtol=1e-10):
            sigma = new
            break
        sigma = new
    chi2 = float(np.sum(((X @ p - logt) / sigma) ** 2))
    return p, chi2


def fit_z(t, xi, xi_err, omega: float = OMEGA, t_min: float = 0.0) -> dict:
    """z from Eq. (5) / (D1) on the points with t >= t_min.  Returns z, b, b', chi2, dof, Q."""
    from scipy.special import gammaincc
    t, xi, xi_err = (np.asarray(a, np.float64) for a in (t, xi, xi_err))
    keep = t >= t_min
    if keep.sum() < 4:
        raise ValueError("need at least 4 points for a 3-parameter fit")
    p, chi2 = _fit_z_once(np.log(t[keep]), xi[keep], xi_err[keep], omega)
    dof = int(keep.sum()) - 3
    return {"z": float(p[0]), "b": float(p[1]), "b1": float(p[2]), "chi2": chi2, "dof": dof,
            "Q": float(gammaincc(dof / 2.0, chi2 / 2.0))}


def fit_z_jackknife(t, C_runs_by_time, omega: float = OMEGA, t_min: float = 0.0) -> dict:
    """C_runs_by_time[time][run, r] -> z with its jackknife error over the runs (App. D):
    xi(t) is recomputed and the fit repeated on every leave-one-out sample."""
    t = np.asarray(t, np.float64)
    stacks = [np.asarray(c, np.float64) for c in C_runs_by_time]
    n = stacks[0].shape[0]
    errs = [c.std(axis=0, ddof=1) / np.sqrt(n) for c in stacks]
    xi_full, xi_err, frozen = [], [], []
    for c in stacks:
        d = {}
        x, e = xi_with_error(c, d)
        xi_full.append(float(x)); xi_err.append(float(e))
        frozen.append({k: d[k] for k in ("r_cut", "r_star", "r_min", "r_max")})
    xi_full, xi_err = np.array(xi_full), np.array(xi_err)
    full = fit_z(t, xi_full, xi_err, omega, t_min)
    import warnings
    zs = []
    with warnings.catch_warnings():
        warnings.simplefilter("ignore", CutoffWarning)            # already reported by xi_with_error
        for i in range(n):
            xi_i = np.array([xi_appendix_c((c.sum(axis=0) - c[i]) / (n - 1), e, cutoffs=f)
                             for c, e, f in zip(stacks, errs, frozen)])
            zs.append(fit_z(t, xi_i, xi_err, omega, t_min)["z"])
    zs = np.array(zs)
    full["z_err"] = float(np.sqrt((n - 1) / n * np.sum((zs - zs.mean()) ** 2)))
    full["xi"], full["xi_err"] = xi_full, xi_err
    return full


# ---- sparse r-grids: cubic-spline interpolation of C(r) ---------------------------
def densify(r, C, C_err=None):
    """C sampled at the sorted separations r (r[0] may be 0) -> (C_dense, err_dense) on r = 0..r[-1].

    The paper measures C(r;t) on a sparse grid of r and integrates with cubic splines (PAPER.md:207,
    ref. [62]); `lattice_measure_list` returns exactly such samples.  The spline goes through
    (0, C(0) = 1 or the given value) and the samples; errors are interpolated linearly."""
    from scipy.interpolate import CubicSpline
    r = np.asarray(r, np.float64)
    C = np.asarray(C, np.float64)
    if r[0] != 0.0:
        r = np.concatenate([[0.0], r])
        C = np.concatenate([[1.0], C])
        if C_err is not None:
            C_err = np.concatenate([[0.0], np.asarray(C_err, np.float64)])
    if np.any(np.diff(r) <= 0):
        raise ValueError("r must be strictly increasing")
    grid = np.arange(int(r[-1]) + 1, dtype=np.float64)
    dense = CubicSpline(r, C)(grid)
    err = None if C_err is None else np.interp(grid, r, np.asarray(C_err, np.float64))
    return dense, err


def xi_sparse(r, C, C_err, details: dict | None = None, **kw) -> float:
    """xi = I_2 / I_1 (App. C) from C(r) on a sparse r-grid: spline to the integers, then xi_appendix_c."""
    dense, err = densify(r, C, C_err)
    return xi_appendix_c(dense, err, details, **kw)


# ---- z from the energy, Eq. (6) / (D2), and the joint fit of Fig. 3 ------------------------------
E_EQ_ISING = -np.sqrt(2.0)     # Onsager: E_eq(T_c) = -sqrt 2
NU_ISING = 1.0                 # D - 1/nu = 1 in two dimensions


def _energy_design(t, z, omega, nu):
    """columns t^(-1/z), t^(-2/z), t^(-(omega + 1/nu)/z) of Eq. (6)."""
    lt = np.log(t)
    return np.stack([np.exp(-lt / z), np.exp(-2.0 * lt / z), np.exp(-(omega + 1.0 / nu) * lt / z)], axis=1)


def _wlsq(X, y, sigma):
    W = 1.0 / sigma
    p, *_ = np.linalg.lstsq(X * W[:, None], y * W, rcond=None)
    return p, float(np.sum(((X @ p - y) * W) ** 2))


def _minimise_over_z(chi2_of_z, bracket=(1.2, 4.0)):
    """The fits are linear in everything but z: minimise the profiled chi^2(z) in one dimension."""
    from scipy.optimize import minimize_scalar
    zs = np.linspace(bracket[0], bracket[1], 57)
    vals = np.array([chi2_of_z(z) for z in zs])
    k = int(np.argmin(vals))
    lo, hi = zs[max(k - 1, 0)], zs[min(k + 1, zs.size - 1)]
    res = minimize_scalar(chi2_of_z, bounds=(lo, hi), method="bounded", options={"xatol": 1e-12})
    return float(res.x)


def fit_z_energy(t, E, E_err, E_eq: float = E_EQ_ISING, omega: float = OMEGA, nu: float = NU_ISING,
                 t_min: float = 0.0) -> dict:
    """z from the local observable: E(t) - E_eq = b t^(-1/z) + b' t^(-2/z) + b'' t^(-(omega+1/nu)/z)
    (Eq. 6 / D2) on the points with t >= t_min.  Only meaningful where E_eq
    is known exactly (Ising: -sqrt 2).  Returns z, b, b1, b2, chi2, dof, Q."""
    from scipy.special import gammaincc
    t, E, E_err = (np.asarray(a, np.float64) for a in (t, E, E_err))
    keep = t >= t_min
    if keep.sum() < 5:
        raise ValueError("need at least 5 points for a 4-parameter fit")
    tt, y, s = t[keep], E[keep] - E_eq, np.maximum(E_err[keep], 1e-300)

    def chi2_of_z(z):
        return _wlsq(_energy_design(tt, z, omega, nu), y, s)[1]

    z = _minimise_over_z(chi2_of_z)
    p, chi2 = _wlsq(_energy_design(tt, z, omega, nu), y, s)
    dof = int(keep.sum()) - 4
    return {"z": z, "b": float(p[0]), "b1": float(p[1]), "b2": float(p[2]), "chi2": chi2, "dof": dof,
            "Q": float(gammaincc(dof / 2.0, chi2 / 2.0))}


def fit_z_joint(datasets, omega: float = OMEGA, nu: float = NU_ISING, t_min: float = 0.0) -> dict:
    """One z for several data sets (the main panel of Fig. 3; "a piecewise function
    that depends on the respective data set").  Each data set is a dict
      {"kind": "xi", "t": ..., "xi": ..., "xi_err": ...}               fitted with Eq. (5) / (D1)
      {"kind": "E",  "t": ..., "E": ..., "E_err": ..., "E_eq": ...}    fitted with Eq. (6) / (D2)
    with its own non-universal amplitudes (b, b' [, b'']); chi^2 is the sum over the sets, the weights
    of the xi sets use the error of xi propagated through f'(xi), iterated."""
    from scipy.special import gammaincc
    sets = []
    for d in datasets:
        t = np.asarray(d["t"], np.float64)
        keep = t >= t_min
        if d["kind"] == "xi":
            xi, xe = np.asarray(d["xi"], np.float64)[keep], np.asarray(d["xi_err"], np.float64)[keep]
            sets.append({"kind": "xi", "logt": np.log(t[keep]), "xi": xi, "xe": xe, "sigma": np.maximum(xe / xi, 1e-300),
                         "npar": 2})
        elif d["kind"] == "E":
            sets.append({"kind": "E", "t": t[keep], "y": np.asarray(d["E"], np.float64)[keep] - d.get("E_eq", E_EQ_ISING),
                         "sigma": np.maximum(np.asarray(d["E_err"], np.float64)[keep], 1e-300), "npar": 3})
        else:
            raise ValueError("kind must be 'xi' or 'E'")
    n_pts = sum(len(s["sigma"]) for s in sets)
    n_par = 1 + sum(s["npar"] for s in sets)
    if n_pts <= n_par:
        raise ValueError("not enough points for the joint fit")

    def solve(z):
        total, pars = 0.0, []
        for s in sets:
            if s["kind"] == "xi":
                X = np.stack([np.ones_like(s["xi"]), s["xi"] ** (-omega)], axis=1)
                p, c2 = _wlsq(X, s["logt"] - z * np.log(s["xi"]), s["sigma"])
            else:
                p, c2 = _wlsq(_energy_design(s["t"], z, omega, nu), s["y"], s["sigma"])
            total += c2
            pars.append(p)
        return total, pars

    z = 2.0
    for _ in range(20):
        z = _minimise_over_z(lambda zz: solve(zz)[0])
        chi2, pars = solve(z)
        changed = False
        for s, p in zip(sets, pars):
            if s["kind"] != "xi":
                continue
            fprime = z / s["xi"] - omega * p[1] * s["xi"] ** (-omega - 1.0)
            new = np.maximum(1e-40 + s["xe"] * np.abs(fprime), 1e-300)       # t_error = 1e-40
            changed = changed or not np.allclose(new, s["sigma"], rtol=1e-10)
            s["sigma"] = new
        if not changed:
            break
    chi2, pars = solve(z)
    dof = n_pts - n_par
    return {"z": z, "amplitudes": [p.tolist() for p in pars], "chi2": chi2, "dof": dof,
            "Q": float(gammaincc(dof / 2.0, chi2 / 2.0))}


def fit_z_energy_jackknife(t, E_runs_by_time, **kw) -> dict:
    """E_runs_by_time[time][run] -> the Eq. (6) fit with jackknife errors over the runs (App. D)."""
    t = np.asarray(t, np.float64)
    stacks = np.array([np.asarray(e, np.float64) for e in E_runs_by_time])      # [time, run]
    n = stacks.shape[1]
    mean, err = stacks.mean(axis=1), stacks.std(axis=1, ddof=1) / np.sqrt(n)
    full = fit_z_energy(t, mean, err, **kw)
    zs = np.array([fit_z_energy(t, (stacks.sum(axis=1) - stacks[:, i]) / (n - 1), err, **kw)["z"] for i in range(n)])
    full["z_err"] = float(np.sqrt((n - 1) / n * np.sum((zs - zs.mean()) ** 2)))
    full["E"], full["E_err"] = mean, err
    return full


# ---- late approach to equilibrium in the two-step protocol, Eq. (8) --------------------------------
def fit_exponential_approach(curves, E_eq: float | None = E_EQ_ISING, t_min: float = 0.0) -> dict:
    """Joint fit of E(t; f) = E_eq + b(f) exp(-t / tau) over several protocols f with one f-independent
    tau (Eq. 8).  curves = [{"f": ..., "t": ..., "E": ..., "E_err": ...}, ...].
    E_eq fixed (Ising: -sqrt 2) or, if None, an additional f-independent parameter (Blume-Capel).
    Linear in b(f) (and E_eq) at fixed tau: the profiled chi^2 is minimised over tau alone."""
    from scipy.optimize import minimize_scalar
    from scipy.special import gammaincc
    cs = []
    for c in curves:
        t = np.asarray(c["t"], np.float64)
        keep = t >= t_min
        cs.append((t[keep], np.asarray(c["E"], np.float64)[keep], np.maximum(np.asarray(c["E_err"], np.float64)[keep], 1e-300)))
    nf = len(cs)
    n_pts = sum(len(c[0]) for c in cs)

    def solve(tau):
        rows, ys, ss = [], [], []
        for k, (t, E, s) in enumerate(cs):
            X = np.zeros((t.size, nf + (1 if E_eq is None else 0)))
            X[:, k] = np.exp(-t / tau)
            if E_eq is None:
                X[:, nf] = 1.0
            rows.append(X); ys.append(E - (0.0 if E_eq is None else E_eq)); ss.append(s)
        p, c2 = _wlsq(np.concatenate(rows), np.concatenate(ys), np.concatenate(ss))
        return c2, p

    t_all = np.concatenate([c[0] for c in cs])
    span = float(t_all.max() - t_all.min()) or 1.0
    taus = np.geomspace(span / 200.0, span * 20.0, 80)
    vals = np.array([solve(x)[0] for x in taus])
    k = int(np.argmin(vals))
    res = minimize_scalar(lambda x: solve(x)[0], bounds=(taus[max(k - 1, 0)], taus[min(k + 1, taus.size - 1)]),
                          method="bounded", options={"xatol": 1e-10 * span})
    tau = float(res.x)
    chi2, p = solve(tau)
    dof = n_pts - (nf + 1 + (1 if E_eq is None else 0))
    return {"tau": tau, "b": {float(c["f"]): float(p[k]) for k, c in enumerate(curves)},
            "E_eq": float(p[nf]) if E_eq is None else float(E_eq), "chi2": chi2, "dof": dof,
            "Q": float(gammaincc(max(dof, 1) / 2.0, chi2 / 2.0))}


def onsager_energy(beta: float) -> float:
    """Exact equilibrium energy per site of the infinite square-lattice Ising model (J = 1, Onsager):
    e = -coth(2 beta) [1 + (2/pi) (2 tanh^2(2 beta) - 1) K(k)],  k = 2 sinh(2 beta) / cosh^2(2 beta),
    K the complete elliptic integral of the first kind.  e(beta_c) = -sqrt 2; the paper
    takes E_eq(T_2) of the two-step protocol from it."""
    from scipy.special import ellipk
    x = 2.0 * beta
    k = 2.0 * np.sinh(x) / np.cosh(x) ** 2
    if abs(1.0 - k) < 1e-14:
        return -np.sqrt(2.0)
    return float(-(1.0 / np.tanh(x)) * (1.0 + (2.0 / np.pi) * (2.0 * np.tanh(x) ** 2 - 1.0) * ellipk(k * k)))
