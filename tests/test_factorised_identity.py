"""The algebra behind the default phi evaluator (include/tnrd.h TNRD_PHI_FACTORED), checked on
the CPU against the oracle's phi (Main Eq. 6 / PAPER.md:553, oracle/tnrd_oracle.c: oracle_phi1):

    exp(-(d - j delta)^2 / 2 gamma^2) = exp(-d^2 / 2 gamma^2) * rho^j * exp(-(j delta)^2 / 2 gamma^2),   rho = exp(delta d / gamma^2)

with d = z - mu_a for the anchor centre mu_a of a group of 13 neighbouring centres, the distance clamped to D = 11.3 scaled
units where the Gaussian factor is taken as zero.  This is a statement about the formula the staging kernel and the fused
kernel implement (csrc/tnrd_internal.h "fact"), written out in numpy double; the CUDA path itself is compared with the
oracle in tests/test_gpu_parity.py."""
import numpy as np
import pytest

import oracle
import tnrd_gen

S, GROUPS, CLAMP = 6, 5, 11.3          # TNRD_FS, TNRD_FG, TNRD_FCLAMP


def factorised_phi(z, w, mu, gamma):
    s = np.sqrt(np.log2(np.e) / (2.0 * gamma * gamma))           # scaled units: 2^{-(s x)^2} = exp(-x^2 / 2 gamma^2)
    delta = (mu[-1] - mu[0]) / (len(mu) - 1)
    ds, kappa = s * delta, 2.0 * s * delta
    out = np.zeros_like(z, dtype=np.float64)
    for g in range(GROUPS):
        a = g * (2 * S + 1) + S
        d = np.clip(s * (z - (mu[0] + a * delta)), -CLAMP, CLAMP)
        gauss = np.where(d * d > 126.0, 0.0, np.exp2(-d * d))    # ex2.approx.ftz flushes below 2^-126
        rho, rhoi = np.exp2(kappa * d), np.exp2(-kappa * d)
        c = lambda j: (w[a + j] if 0 <= a + j < len(mu) else 0.0) * np.exp2(-(j * ds) ** 2)
        h = np.full_like(z, c(S), dtype=np.float64)
        for j in range(S - 1, -1, -1):
            h = h * rho + c(j)
        hl = np.full_like(z, c(-S), dtype=np.float64)
        for j in range(-S + 1, 0):
            hl = hl * rhoi + c(j)
        out += gauss * (hl * rhoi + h)
    return out


@pytest.mark.parametrize("gamma", [10.0, 9.6, 14.0, 30.0])
def test_factorised_form_is_the_oracle_phi(gamma):
    prm = tnrd_gen.make_params(11, 1, 6, 5)
    mu = prm["rbf_mu"].astype(np.float64)
    r = np.random.default_rng([150305768, 99])
    z = np.concatenate([r.uniform(-420.0, 420.0, 4000), mu, mu + 5.0, [-1000.0, 1000.0, 0.0]])
    for i in range(6):
        w = prm["rbf_w"][0, i].astype(np.float64)
        want = oracle.phi(z, w, mu, gamma)
        got = factorised_phi(z, w, mu, gamma)
        # the only difference is the mass of the terms taken as zero beyond the clamp: each below 2^-(D - S delta')^2 of its
        # weight (2^-38 for gamma = delta; the staging kernel requires at least 2^-30)
        ds = np.sqrt(np.log2(np.e) / 2.0) * (mu[1] - mu[0]) / gamma
        dropped = 2.0 ** -((CLAMP - S * ds) ** 2)
        assert dropped <= 2.0 ** -30
        assert np.max(np.abs(got - want)) <= 4.0 * dropped * np.max(np.abs(w)) + 1e-15, (gamma, i)


def test_range_conditions_of_the_default_centres():
    """gamma = delta: rho^j 2^{-(j delta')^2} stays below 2^92 at the clamp and the nearest dropped term is 6.2 scaled units
    away (the two numbers the staging kernel checks on the device; DESIGN.md quotes 89.2 and 38.4)."""
    ds = np.sqrt(np.log2(np.e) / 2.0)
    emax = max(j * 2.0 * ds * CLAMP - (j * ds) ** 2 for j in range(1, S + 1))
    reach = CLAMP - S * ds
    assert abs(emax - 89.2) < 0.1 and emax <= 92.0
    assert abs(reach ** 2 - 38.4) < 0.1 and reach ** 2 >= 30.0
    assert GROUPS * (2 * S + 1) >= 63 and (GROUPS - 1) * (2 * S + 1) + S < 63      # every centre in exactly one group
