"""Filter bounds [a, b] for synthetic runs: a k-step Lanczos estimate (harness helper).

PAPER.md:469 takes lambda_max, lambda_min from Lanczos and lambda_T from the previous SCF iteration's
Rayleigh quotients; a synthetic run has no previous SCF, so a = theta_min + fw (b - theta_min) stands in
(SURVEY 8(c) O10 / reading A15). a and b are INPUTS of the filter on both the CUDA path and the oracle,
so this is input generation, not part of either implementation; it only calls the `apply_H` it is given.
"""
import numpy as np

from .synth import random_block


def lanczos_bounds(apply_H, nrows, k=20, seed=7, fw=0.02):
    """Filter bounds [a, b] from a k-step Lanczos run on Hhat (harness helper).

    `apply_H` maps a complex128 [nrows, 1] host array to Hhat times it. Returns (a, b, theta_min, theta_max):
    b = theta_max + |beta_k| is a safe upper bound, a = theta_min + fw (b - theta_min) stands in for lambda_T.
    The filter takes a and b as inputs, so parity between the CUDA path and the oracle never depends on this.
    """
    rng = np.random.Generator(np.random.PCG64(seed))
    v = random_block(rng, nrows, 1); v /= np.linalg.norm(v)
    vprev = np.zeros_like(v); beta = 0.0
    alphas, betas = [], []
    for _ in range(k):
        w = apply_H(v) - beta * vprev
        alpha = float(np.real(np.vdot(v, w)))
        w = w - alpha * v
        beta = float(np.linalg.norm(w))
        alphas.append(alpha); betas.append(beta)
        if beta < 1e-14:
            break
        vprev, v = v, w / beta
    T = np.diag(alphas) + np.diag(betas[:-1], 1) + np.diag(betas[:-1], -1)
    th = np.linalg.eigvalsh(T)
    b = float(th[-1] + abs(betas[-1])); tmin = float(th[0])
    a = tmin + fw * (b - tmin)
    return a, b, tmin, float(th[-1])
