"""Writes the expected values of tests/golden/closed_form_quadrature.txt.

Integrates the UN-marginalised likelihood of Eq. 8,
    L(N, mu, lambda) = (2 pi lambda^2)^(-n/2) exp(-sum_r (I_obs(r) - N I_calc(r) + mu)^2 / (2 lambda^2)),
over N, mu in R and lambda > 0 with unit priors (reading R1) by brute-force quadrature: for each lambda a 2-D
trapezoid rule in (N, mu) on the raw sum of squares (no completed squares: that algebra is what the closed form
under test relies on), then a trapezoid rule in u = log(lambda).  It imports nothing from oracle/ or the CUDA package.

    python tests/golden/make_closed_form_golden.py          # rewrites the data lines of the fixture
"""
from pathlib import Path

import numpy as np

CASES = [
    ([0.3, -1.2, 0.8, 2.1, -0.5, 0.0, 1.4, -0.9, 0.6], [0.1, -0.4, 0.5, 1.0, -0.2, 0.3, 0.7, -0.6, 0.2]),
    ([1.0, 2.0, -1.0, 0.5, 0.25, -2.0, 3.0, 0.0, 1.5, -0.75, 0.1, 0.9], [0.2, 0.9, -0.3, 0.0, 0.4, -1.1, 1.2, 0.1, 0.8, -0.2, -0.1, 0.5]),
    ([5.0, 4.0, 6.5, 5.5, 3.0, 4.5, 7.0, 5.2, 6.1, 4.4, 5.9, 3.8, 6.6, 5.1, 4.9, 5.3],
     [-0.5, -1.0, 0.4, 0.1, -1.6, -0.8, 0.9, -0.2, 0.5, -0.9, 0.2, -1.2, 0.6, 0.0, -0.3, -0.1]),
]


def log_integral(io, ic, nodes=401, n_lam=1201):
    io, ic = np.asarray(io, float), np.asarray(ic, float)
    n = io.size
    # centre and widths of the Gaussian in (N, mu) -- only used to PLACE the quadrature nodes
    G = np.array([[np.sum(ic * ic), -np.sum(ic)], [-np.sum(ic), float(n)]])
    rhs = np.array([np.sum(io * ic), -np.sum(io)])
    Ns, mus = np.linalg.solve(G, rhs)
    E = np.sum((io - Ns * ic + mus) ** 2)
    cov = np.linalg.inv(G)
    us = np.linspace(np.log(1e-3 * np.sqrt(E / n)), np.log(1e3 * np.sqrt(E / n)), n_lam)
    logf = np.empty_like(us)
    for i, u in enumerate(us):
        lam = np.exp(u)
        wN, wm = 12.0 * lam * np.sqrt(cov[0, 0]), 12.0 * lam * np.sqrt(cov[1, 1])
        Ng = np.linspace(Ns - wN, Ns + wN, nodes)
        mg = np.linspace(mus - wm, mus + wm, nodes)
        NN, MM = np.meshgrid(Ng, mg, indexing="ij")
        S = np.zeros_like(NN)
        for r in range(n):                                    # the raw sum of squares of Eq. 8 at every node
            S += (io[r] - NN * ic[r] + MM) ** 2
        ex = -S / (2 * lam * lam)
        mx = ex.max()
        w = np.exp(ex - mx)
        integral = np.trapezoid(np.trapezoid(w, mg, axis=1), Ng)
        logf[i] = np.log(integral) + mx - 0.5 * n * np.log(2 * np.pi * lam * lam) + u      # d lambda = lambda du
    mx = logf.max()
    return float(mx + np.log(np.trapezoid(np.exp(logf - mx), us)))


def main():
    path = Path(__file__).with_name("closed_form_quadrature.txt")
    head = [ln for ln in path.read_text().splitlines() if ln.startswith("#")]
    rows = []
    for io, ic in CASES:
        v = log_integral(io, ic)
        rows.append(f"{len(io)} {' '.join(repr(x) for x in io)} | {' '.join(repr(x) for x in ic)} | {v:.10f}")
    path.write_text("\n".join(head + rows) + "\n")
    print("\n".join(rows))


if __name__ == "__main__":
    main()
