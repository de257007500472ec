"""Pins of the CPU oracle against what the paper and the mathematics fix (CPU only).

Each test names the passage of /root/reference/PAPER.md (or the DESIGN.md reading) it pins.
None of the expected values comes from the CUDA path.
"""
import math
import os

import numpy as np
import pytest

import gf_inputs as gi
import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
SUBGROUPS = [(0, 1), (0, 2), (1, 2)]


def su2_matrix(a):
    """The paper-side SU(2) parametrisation used by reading A4."""
    return np.array([[a[0] + 1j * a[3], a[2] + 1j * a[1]],
                     [-a[2] + 1j * a[1], a[0] - 1j * a[3]]])


def embed(a, i, j):
    E = np.eye(3, dtype=complex)
    m = su2_matrix(a)
    E[i, i], E[i, j], E[j, i], E[j, j] = m[0, 0], m[0, 1], m[1, 0], m[1, 1]
    return E


def random_unit4(rng, n):
    a = rng.standard_normal((n, 4))
    return a / np.linalg.norm(a, axis=1, keepdims=True)


# ------------------------------------------------------------------------------- Philox

def test_philox_known_answers():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt"))
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        w = [int(x, 16) for x in r]
        assert oracle.philox4x32_10(w[0:4], w[4:6]) == tuple(w[6:10])


def test_site_uniforms_are_24_bit_fractions_of_the_philox_words():
    seed, ctr, s = 0x299f31d0a4093822, 0x13198a2e, 0x85a308d3243f6a88
    # third golden vector: counter (s_lo, s_hi, ctr, 0) differs from it only in word 3
    words = oracle.philox4x32_10([s & 0xffffffff, s >> 32, ctr, 0], [seed & 0xffffffff, seed >> 32])
    u = oracle.site_uniforms(seed, ctr, s)
    for k in range(3):
        assert u[k] == (words[k] >> 8) / 2.0 ** 24
        assert 0.0 <= u[k] < 1.0


def test_site_uniforms_keep_all_24_leading_bits():
    """Reading A8 / SURVEY O4: u_k = (word_k >> 8) * 2^-24 -- the top 24 bits, bit 8 included (a 23-bit
    fraction (w >> 9) * 2^-23 agrees whenever bit 8 is clear, as in the golden vector above), from words
    0, 1, 2 in that order of the counter (s_lo, s_hi, half-sweep counter, 0) under the key (seed_lo, seed_hi)."""
    rng = np.random.default_rng(41)
    bit8 = [0, 0, 0]
    for _ in range(100):
        seed = int(rng.integers(0, 2 ** 63)) * 2 + int(rng.integers(0, 2))
        ctr = int(rng.integers(0, 2 ** 32))
        s = int(rng.integers(0, 2 ** 40))
        words = oracle.philox4x32_10([s & 0xffffffff, s >> 32, ctr, 0], [seed & 0xffffffff, seed >> 32])
        u = oracle.site_uniforms(seed, ctr, s)
        for k in range(3):
            assert u[k] == (words[k] >> 8) / 2.0 ** 24
            assert u[k] * 2 ** 24 == float(words[k] >> 8)          # a 24-bit integer, exactly
            bit8[k] += (words[k] >> 8) & 1
    assert all(20 < b < 80 for b in bit8)                          # the lowest kept bit is set about half the time
    # all-ones site, counter and seed: the high words of s and of the seed are used
    u = oracle.site_uniforms(0xffffffffffffffff, 0xffffffff, 0xffffffffffffffff)
    w3 = oracle.philox4x32_10([0xffffffff] * 3 + [0], [0xffffffff] * 2)
    assert list(u) == [(w >> 8) / 2.0 ** 24 for w in w3[:3]]


# ------------------------------------------------- eq. 9: the SU(2) closed form

def test_eq9_literal_for_an_su2_block():
    """K_sub = r W, W in SU(2): eq. 9 g = K^dagger / sqrt(det K^dagger) = W^dagger."""
    rng = np.random.default_rng(1)
    for (i, j) in SUBGROUPS:
        W = su2_matrix(random_unit4(rng, 1)[0])
        r = 0.3 + 3.0 * rng.random()
        K = rng.standard_normal((3, 3)) + 1j * rng.standard_normal((3, 3))
        K[np.ix_([i, j], [i, j])] = r * W
        Kb = K[np.ix_([i, j], [i, j])]
        g9 = Kb.conj().T / np.sqrt(np.linalg.det(Kb.conj().T))       # eq. 9 as printed
        a = oracle.su2_update(oracle.su2_vector(K, i, j), oracle.RELAX)
        assert np.allclose(su2_matrix(a), g9, atol=1e-14)
        assert np.allclose(su2_matrix(a), W.conj().T, atol=1e-14)


def test_su2_closed_form_beats_brute_force():
    """the closed form maximises Re tr[g K] over the SU(2) subgroup; no random
    SU(2) element and no local perturbation does better, and the maximum is |v| + Re K_kk."""
    rng = np.random.default_rng(2)
    for trial in range(6):
        K = rng.standard_normal((3, 3)) + 1j * rng.standard_normal((3, 3))
        for (i, j) in SUBGROUPS:
            k = 3 - i - j
            v = oracle.su2_vector(K, i, j)
            a = oracle.su2_update(v, oracle.RELAX)
            assert abs(np.linalg.norm(a) - 1.0) < 1e-15
            best = np.trace(embed(a, i, j) @ K).real
            assert abs(best - (np.linalg.norm(v) + K[k, k].real)) < 1e-13
            cand = random_unit4(rng, 20000)
            local = a + 1e-3 * rng.standard_normal((2000, 4))
            local /= np.linalg.norm(local, axis=1, keepdims=True)
            for c in np.concatenate([cand, local]):
                # Re tr[E K] written out for the 2x2 block plus the untouched diagonal entry
                m = su2_matrix(c)
                val = (m[0, 0] * K[i, i] + m[0, 1] * K[j, i] + m[1, 0] * K[i, j] + m[1, 1] * K[j, j]).real \
                    + K[k, k].real
                assert val <= best + 1e-12
            # spot check of the written-out trace against the full matrix product
            assert abs(val - np.trace(embed(c, i, j) @ K).real) < 1e-12


def test_site_g_is_the_ordered_product_of_three_subgroup_maximisers():
    """PAPER.md:76 with readings A5/A6: g = E3 E2 E1, each E_k maximising Re tr[E K_k] for the
    refreshed K_k; every step cannot decrease Re tr[g K]; g is in SU(3)."""
    rng = np.random.default_rng(3)
    K = rng.standard_normal((3, 3)) + 1j * rng.standard_normal((3, 3))
    g = oracle.site_g(K, oracle.RELAX)
    Kc, gc, f_prev = K.copy(), np.eye(3, dtype=complex), np.trace(K).real
    for (i, j) in SUBGROUPS:
        E = embed(oracle.su2_update(oracle.su2_vector(Kc, i, j), oracle.RELAX), i, j)
        Kc, gc = E @ Kc, E @ gc
        f = np.trace(gc @ K).real
        assert f >= f_prev - 1e-13
        f_prev = f
    assert np.allclose(g, gc, atol=1e-14)
    assert np.allclose(g @ g.conj().T, np.eye(3), atol=1e-14)
    assert abs(np.linalg.det(g) - 1) < 1e-14


def test_site_g_composition_with_overrelaxation_and_stochastic_draws():
    """Readings A5-A8 for the variants of PAPER.md:80 and :84: EVERY one of the three SU(2) factors is
    overrelaxed with the same omega, and subgroup k takes the draw u_k -- pinned against the ordered numpy
    product of the separately pinned su2_vector / su2_update steps, with three different draws straddling p."""
    rng = np.random.default_rng(30)
    for trial in range(4):
        K = rng.standard_normal((3, 3)) + 1j * rng.standard_normal((3, 3))
        cases = [(oracle.OVERRELAX, 1.7, 0.0, (0.0, 0.0, 0.0))]
        # every pattern of "square / do not square" over the three subgroups
        for mask in range(8):
            cases.append((oracle.STOCHASTIC, 1.0, 0.5, tuple(0.1 if mask >> k & 1 else 0.9 for k in range(3))))
        seen = []
        for algo, omega, p, u in cases:
            g = oracle.site_g(K, algo, omega, p, u)
            Kc, gc = K.copy(), np.eye(3, dtype=complex)
            for k, (i, j) in enumerate(SUBGROUPS):
                E = embed(oracle.su2_update(oracle.su2_vector(Kc, i, j), algo, omega, p, u[k]), i, j)
                Kc, gc = E @ Kc, E @ gc
            assert np.allclose(g, gc, atol=1e-14), (algo, u)
            assert np.allclose(g @ g.conj().T, np.eye(3), atol=1e-14) and abs(np.linalg.det(g) - 1) < 1e-14
            seen.append(g)
        for a in range(len(seen)):                       # all nine variants really are different updates
            for b in range(a + 1, len(seen)):
                assert np.abs(seen[a] - seen[b]).max() > 1e-3


def test_site_g_closed_form_per_subgroup_on_a_real_rotation():
    """K = a real rotation by phi embedded in ONE subgroup (i,j): the other two subgroups see a real diagonal
    block, i.e. v proportional to (1,0,0,0), and do nothing, so g must be exactly the embedded SU(2) answer:
      relaxation (eq. 9):        rotation by -phi  (g K = 1)
      overrelaxation (A7):       rotation by -phi', tan phi' = omega sin phi / (omega cos phi + 1 - omega)
      stochastic (A8), u_k < p:  rotation by -2 phi; u_k >= p: rotation by -phi,
    whichever of the three subgroups it is -- also the last one -- and whatever the OTHER two draws are."""
    omega, p = 1.7, 0.5
    for k, (i, j) in enumerate(SUBGROUPS):
        for phi in (0.3, -0.8, 1.2):
            def rot(angle):
                R = np.eye(3, dtype=complex)
                R[i, i] = R[j, j] = math.cos(angle)
                R[i, j], R[j, i] = math.sin(angle), -math.sin(angle)
                return R
            K = 2.5 * rot(phi)
            assert np.allclose(oracle.site_g(K, oracle.RELAX), rot(-phi), atol=1e-15)
            phi_or = math.atan2(omega * math.sin(phi), omega * math.cos(phi) + 1 - omega)
            assert abs(phi_or) > abs(phi) * 1.2                      # it does overshoot
            assert np.allclose(oracle.site_g(K, oracle.OVERRELAX, omega), rot(-phi_or), atol=1e-15)
            others_low = [0.9] * 3
            others_low[k] = 0.1                                      # only subgroup k squares
            assert np.allclose(oracle.site_g(K, oracle.STOCHASTIC, 1.0, p, others_low), rot(-2 * phi), atol=1e-15)
            others_high = [0.1] * 3
            others_high[k] = 0.9                                     # every subgroup but k squares (the identity)
            assert np.allclose(oracle.site_g(K, oracle.STOCHASTIC, 1.0, p, others_high), rot(-phi), atol=1e-15)


def test_zero_K_gives_identity():
    """Reading A9."""
    assert np.array_equal(oracle.site_g(np.zeros((3, 3), complex), oracle.OVERRELAX, 1.7), np.eye(3))


# -------------------------------------------------- section 3.1 / 3.2 variants

def test_overrelaxation_is_first_order_g_to_the_omega():
    """Reading A7: omega = 1 is eq. 9; the rotation angle phi' of the update agrees with the exact
    a^omega (angle omega*phi) to first order: (phi' - omega phi)/phi^3 -> -omega(2 omega-1)(omega-1)/6."""
    axis = np.array([0.3, -0.5, 0.81])
    axis /= np.linalg.norm(axis)
    for omega in (1.0, 1.3, 1.7, 1.95):
        for phi in (1e-1, 3e-2, 1e-2):
            v = 2.7 * np.concatenate([[math.cos(phi)], math.sin(phi) * axis])
            a = oracle.su2_update(v, oracle.OVERRELAX, omega)
            assert abs(np.linalg.norm(a) - 1) < 1e-15
            assert np.allclose(a[1:] / np.linalg.norm(a[1:]), axis, atol=1e-12)   # same axis
            phi_new = math.atan2(np.linalg.norm(a[1:]), a[0])
            coeff = (phi_new - omega * phi) / phi ** 3
            assert abs(coeff - (-omega * (2 * omega - 1) * (omega - 1) / 6)) < 0.02 + 2 * phi ** 2
        v = np.array([0.4, -1.1, 0.7, 2.0])
        assert np.array_equal(oracle.su2_update(v, oracle.OVERRELAX, 1.0), oracle.su2_update(v, oracle.RELAX))


def test_stochastic_step_squares_with_probability_p():
    """g -> g^2 with probability p; u < p decides (reading A8)."""
    rng = np.random.default_rng(4)
    v = rng.standard_normal(4)
    a = oracle.su2_update(v, oracle.RELAX)
    sq = su2_matrix(a) @ su2_matrix(a)
    assert np.allclose(su2_matrix(oracle.su2_update(v, oracle.STOCHASTIC, p=0.8, u=0.79)), sq, atol=1e-15)
    assert np.array_equal(oracle.su2_update(v, oracle.STOCHASTIC, p=0.8, u=0.8), a)
    assert np.array_equal(oracle.su2_update(v, oracle.STOCHASTIC, p=0.0, u=0.0), a)
    # the draws themselves: the fraction below p tends to p
    u = np.array([oracle.site_uniforms(2013, 7, s) for s in range(4000)]).ravel()
    assert abs((u < 0.8).mean() - 0.8) < 0.02
    assert abs(u.mean() - 0.5) < 0.02


# ---------------------------------------------------------------- F and theta (eq. 2, 4, 5, 6)

DIMS = (4, 6, 8, 4)   # asymmetric on purpose: index mistakes show


def test_unit_links_F_is_1_theta_is_0_sweep_is_identity():
    U = gi.unit_links(DIMS)
    for gauge in (oracle.LANDAU, oracle.COULOMB):
        assert np.all(np.asarray(oracle.functional(U, DIMS, gauge)) == 1.0)
        assert np.all(np.asarray(oracle.theta(U, DIMS, gauge)) == 0.0)
        V = U.copy()
        for parity in (0, 1):
            oracle.sweep(V, DIMS, parity, gauge, oracle.OVERRELAX, 1.7)
        assert np.array_equal(U, V)
    assert oracle.plaquette(U, DIMS) == 1.0


def test_functional_eq2_equals_eq6():
    """PAPER.md:39 vs :60: F = 1/(2 Nc Nd V) Re sum_x tr K(x) (g = 1)."""
    U = gi.smooth_random_gauge(DIMS, 0.4, 11)
    V = int(np.prod(DIMS))
    sumK = sum(np.trace(oracle.site_K(U, DIMS, s)).real for s in range(V))
    assert abs(oracle.functional(U, DIMS) - sumK / (2 * 3 * 4 * V)) < 1e-14
    # and eq. 2 itself with a library reduction
    assert abs(oracle.functional(U, DIMS) - np.trace(U, axis1=-2, axis2=-1).real.sum() / (3 * 4 * V)) < 1e-14
    # Coulomb, reading A2: per slice over the spatial links
    Fc = oracle.functional(U, DIMS, oracle.COULOMB)
    ref = np.trace(U[:, :, :, :, 1:], axis1=-2, axis2=-1).real.sum(axis=(1, 2, 3, 4)) / (3 * 3 * V / DIMS[0])
    assert np.allclose(Fc, ref, atol=1e-14)


def test_theta_closed_form_for_an_abelian_wave():
    """eq. 4-5 with reading A1 on U_mu(x) = exp(i a_mu(x_mu) T), T = diag(1,-1,0): A_mu = sin(a_mu) T
    exactly, cross terms between directions telescope away, so
    theta = 2/(3V) sum_mu (V/N_mu) sum_{x_mu} (sin a_mu(x_mu) - sin a_mu(x_mu - 1))^2."""
    nt, nx, ny, nz = DIMS
    amp = (0.7, 0.3, 1.1, 0.5)
    wave = (1, 2, 3, 1)
    n_of_mu = DIMS
    U = np.zeros(gi.field_shape(DIMS) + (4, 3, 3), complex)
    coords = np.meshgrid(np.arange(nt), np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    coord_of_mu = (coords[0], coords[3], coords[2], coords[1])

    def a_of(mu, c):
        return amp[mu] * np.cos(2 * np.pi * wave[mu] * c / n_of_mu[mu] + 0.37 * mu)

    for mu in range(4):
        a = a_of(mu, coord_of_mu[mu])
        U[..., mu, 0, 0], U[..., mu, 1, 1], U[..., mu, 2, 2] = np.exp(1j * a), np.exp(-1j * a), 1.0
    V = nt * nx * ny * nz

    def one_d(mu):
        c = np.arange(n_of_mu[mu])
        return ((np.sin(a_of(mu, c)) - np.sin(a_of(mu, c - 1))) ** 2).sum()

    expect = 2.0 / (3 * V) * sum(V / n_of_mu[mu] * one_d(mu) for mu in range(4))
    assert abs(oracle.theta(U, DIMS) - expect) < 1e-14
    th_c = oracle.theta(U, DIMS, oracle.COULOMB)          # reading A17: spatial directions, per slice
    Vs = V // nt
    expect_c = 2.0 / (3 * Vs) * sum(Vs / n_of_mu[mu] * one_d(mu) for mu in (1, 2, 3))
    assert np.allclose(th_c, expect_c, atol=1e-14)


def test_theta_small_field_limit_and_direction_convention():
    """A_mu = eps H_mu + O(eps^3) for U = exp(i eps H): theta/eps^2 -> 1/(3V) sum_x |sum_mu (H_mu(x)
    - H_mu(x - mu))|^2, with the backward difference of eq. 4."""
    eps = 1e-4
    U, H = gi.smooth_links(DIMS, eps, 5)
    div = sum(H[..., mu, :, :] - np.roll(H[..., mu, :, :], +1, axis=gi.AXIS_OF_MU[mu]) for mu in range(4))
    expect = (np.abs(div) ** 2).sum() / (3 * np.prod(DIMS))
    assert abs(oracle.theta(U, DIMS) / eps ** 2 / expect - 1) < 1e-6
    fwd = sum(np.roll(H[..., mu, :, :], -1, axis=gi.AXIS_OF_MU[mu]) - H[..., mu, :, :] for mu in range(4))
    # the per-site Delta is the BACKWARD divergence at that site, not the forward one
    s = 137
    D = oracle.site_delta(U, DIMS, s) / eps
    assert np.allclose(D, div.reshape(-1, 3, 3)[s], atol=1e-6)
    assert not np.allclose(D, fwd.reshape(-1, 3, 3)[s], atol=1e-2)


def test_theta_from_links_equals_theta_from_K():
    """Delta(x) = traceless[(K - K^dagger)/2i]: ties eq. 4 to eq. 8 (same neighbours, same signs)."""
    U = gi.smooth_random_gauge(DIMS, 0.5, 6)
    for gauge in (oracle.LANDAU, oracle.COULOMB):
        for s in (0, 1, 77, 500, int(np.prod(DIMS)) - 1):
            K = oracle.site_K(U, DIMS, s, gauge)
            D = (K - K.conj().T) / 2j
            D -= np.trace(D) / 3 * np.eye(3)
            assert np.allclose(D, oracle.site_delta(U, DIMS, s, gauge), atol=1e-14)


def test_F_and_theta_invariant_under_a_global_rotation():
    U = gi.smooth_random_gauge(DIMS, 0.5, 7)
    h = gi.haar_su3(np.random.default_rng(8), ())
    Uh = np.ascontiguousarray(np.einsum("ab,...bc,dc->...ad", h, U, h.conj()))
    assert abs(oracle.functional(U, DIMS) - oracle.functional(Uh, DIMS)) < 1e-14
    assert abs(oracle.theta(U, DIMS) / oracle.theta(Uh, DIMS) - 1) < 1e-12


# --------------------------------------------------------------------------- the sweep

def test_plaquette_is_gauge_invariant_and_links_stay_in_SU3():
    U0, _ = gi.smooth_links(DIMS, 0.6, 9)
    P0 = oracle.plaquette(U0, DIMS)
    assert 0.0 < P0 < 1.0
    U = np.ascontiguousarray(gi.gauge_transform(U0, gi.random_gauge(DIMS, 10)))
    assert abs(oracle.plaquette(U, DIMS) - P0) < 1e-14          # pins the plaquette itself
    variants = [(oracle.LANDAU, oracle.RELAX, 1.0, 0.0), (oracle.LANDAU, oracle.OVERRELAX, 1.7, 0.0),
                (oracle.LANDAU, oracle.STOCHASTIC, 1.0, 0.8), (oracle.COULOMB, oracle.OVERRELAX, 1.7, 0.0),
                (oracle.COULOMB, oracle.STOCHASTIC, 1.0, 0.8)]
    for gauge, algo, omega, p in variants:
        W = U.copy()
        for it in range(5):
            for parity in (0, 1):
                oracle.sweep(W, DIMS, parity, gauge, algo, omega, p, seed=2013, half_sweep_counter=2 * it + parity)
        assert abs(oracle.plaquette(W, DIMS) - P0) < 1e-12
        d_unit, d_det = oracle.unitarity_defect(W, DIMS)
        assert d_unit < 1e-12 and d_det < 1e-12
        assert not np.allclose(W, U)


def test_unitarity_defect_on_links_with_a_known_defect():
    """SURVEY 8(c) O6 / acceptance (4): out[0] = max_{links, entries} |U U^dagger - 1|, out[1] = max |det U - 1|,
    on fields whose defect is known in closed form -- the checker behind every "links stay in SU(3)" assertion.
      U -> (1 + d) U:            U U^dagger - 1 = (2d + d^2) 1,    det = (1 + d)^3
      two rows swapped:          still unitary,                    det = -1
      U -> e^{i phi} U:          still unitary,                    det = e^{3 i phi}, |det - 1| = 2 |sin(3 phi / 2)|
      U = 1 + e E_01 (shear):    U U^dagger - 1 = e (E_01 + E_10) + e^2 E_00,  det = 1
    each planted on a single link (first, last, middle, any mu) of an otherwise exact SU(3) field."""
    dims = (4, 4, 6, 2)
    U0 = gi.hot_links(dims, 77)
    base = oracle.unitarity_defect(U0, dims)
    assert base[0] < 1e-14 and base[1] < 1e-14
    flat_shape = (-1, 4, 3, 3)
    V = int(np.prod(dims))
    spots = [(0, 0), (V - 1, 3), (V // 2 + 3, 1), (17, 2)]
    d = 1e-3
    for s, mu in spots:
        U = U0.copy()
        U.reshape(flat_shape)[s, mu] *= 1 + d
        du, dd = oracle.unitarity_defect(U, dims)
        assert abs(du - (2 * d + d * d)) < 1e-14 and abs(dd - ((1 + d) ** 3 - 1)) < 1e-14
        U = U0.copy()
        L = U.reshape(flat_shape)[s, mu]
        L[[0, 1]] = L[[1, 0]]
        du, dd = oracle.unitarity_defect(U, dims)
        assert du < 1e-14 and abs(dd - 2.0) < 1e-14
        U = U0.copy()
        phi = 0.2
        U.reshape(flat_shape)[s, mu] *= np.exp(1j * phi)
        du, dd = oracle.unitarity_defect(U, dims)
        assert du < 1e-14 and abs(dd - 2 * abs(math.sin(1.5 * phi))) < 1e-14
        U = U0.copy()
        e = 0.25
        shear = np.eye(3, dtype=complex)
        shear[0, 1] = e
        U.reshape(flat_shape)[s, mu] = shear
        du, dd = oracle.unitarity_defect(U, dims)
        assert abs(du - e) < 1e-15 and dd < 1e-14          # dd: the rounding of the other (Haar) links
    # the two outputs are maxima over all links, independently: two different links carry the two worst defects
    U = U0.copy()
    U.reshape(flat_shape)[5, 0] *= 1 + d
    U.reshape(flat_shape)[9, 3] *= np.exp(0.4j)
    du, dd = oracle.unitarity_defect(U, dims)
    assert abs(du - (2 * d + d * d)) < 1e-14 and abs(dd - 2 * math.sin(0.6)) < 1e-14
    # and against a library routine on a generically perturbed field
    rng = np.random.default_rng(78)
    U = U0 + 1e-3 * (rng.standard_normal(U0.shape) + 1j * rng.standard_normal(U0.shape))
    du, dd = oracle.unitarity_defect(np.ascontiguousarray(U), dims)
    UUd = np.einsum("...ab,...cb->...ac", U, U.conj()) - np.eye(3)
    assert abs(du - np.abs(UUd).max()) < 1e-15
    assert abs(dd - np.abs(np.linalg.det(U) - 1).max()) < 1e-15
    assert du > 1e-3 and dd > 1e-4


def test_F_non_decreasing_under_relaxation():
    """the sweep optimises F locally; at omega = 1 every half-sweep raises F."""
    for gauge in (oracle.LANDAU, oracle.COULOMB):
        U = gi.smooth_random_gauge(DIMS, 0.5, 12)
        F = np.asarray(oracle.functional(U, DIMS, gauge))
        assert np.all(F < 0.5)                                   # a random gauge is far from the maximum
        for it in range(6):
            for parity in (0, 1):
                oracle.sweep(U, DIMS, parity, gauge, oracle.RELAX)
                Fn = np.asarray(oracle.functional(U, DIMS, gauge))
                assert np.all(Fn >= F - 1e-15)
                F = Fn
        assert np.all(F > 0.6)


def test_p1_stochastic_sweep_is_microcanonical():
    """g^2 applied with p = 1 leaves Re tr[a K_sub] and hence F unchanged (reading A8)."""
    U = gi.smooth_random_gauge(DIMS, 0.5, 13)
    F0 = oracle.functional(U, DIMS)
    W = U.copy()
    for it in range(5):
        for parity in (0, 1):
            oracle.sweep(W, DIMS, parity, oracle.LANDAU, oracle.STOCHASTIC, 1.0, 1.0, 99, 2 * it + parity)
    assert abs(oracle.functional(W, DIMS) - F0) < 1e-13
    assert not np.allclose(W, U)
    # p = 0 is plain relaxation, bit for bit
    A, B = U.copy(), U.copy()
    oracle.sweep(A, DIMS, 0, oracle.LANDAU, oracle.STOCHASTIC, 1.0, 0.0, 99, 0)
    oracle.sweep(B, DIMS, 0, oracle.LANDAU, oracle.RELAX)
    assert np.array_equal(A, B)


def test_su2_embedded_field_is_fixed_exactly_on_the_updated_parity():
    """The SU(2) textbook case of eq. 9: links in one SU(2) subgroup -> after one omega = 1
    half-sweep Delta(x) = 0 on the updated parity."""
    rng = np.random.default_rng(14)
    a = random_unit4(rng, int(np.prod(DIMS)) * 4).reshape(gi.field_shape(DIMS) + (4, 4))
    U = np.zeros(gi.field_shape(DIMS) + (4, 3, 3), complex)
    U[..., 2, 2] = 1.0
    U[..., 0, 0], U[..., 0, 1] = a[..., 0] + 1j * a[..., 3], a[..., 2] + 1j * a[..., 1]
    U[..., 1, 0], U[..., 1, 1] = -a[..., 2] + 1j * a[..., 1], a[..., 0] - 1j * a[..., 3]
    oracle.sweep(U, DIMS, 1, oracle.LANDAU, oracle.RELAX)
    nt, nx, ny, nz = DIMS
    worst_on, worst_off = 0.0, 0.0
    for s in range(0, int(np.prod(DIMS)), 7):
        x, y, z, t = s % nx, (s // nx) % ny, (s // (nx * ny)) % nz, s // (nx * ny * nz)
        d = np.abs(oracle.site_delta(U, DIMS, s)).max()
        if (x + y + z + t) % 2 == 1:
            worst_on = max(worst_on, d)
        else:
            worst_off = max(worst_off, d)
    assert worst_on < 1e-14 and worst_off > 1e-2


def test_sweep_result_is_independent_of_the_visiting_order():
    """same-parity sites share no link, so any order gives the same bits."""
    U = gi.smooth_random_gauge(DIMS, 0.5, 15)
    for gauge in (oracle.LANDAU, oracle.COULOMB):
        A, B = U.copy(), U.copy()
        for parity in (0, 1):
            oracle.sweep(A, DIMS, parity, gauge, oracle.STOCHASTIC, 1.0, 0.7, 5, parity)
            oracle.sweep(B, DIMS, parity, gauge, oracle.STOCHASTIC, 1.0, 0.7, 5, parity, reverse_order=True)
        assert np.array_equal(A, B)
    n = oracle.set_threads(3)
    try:
        C = U.copy()
        for parity in (0, 1):
            oracle.sweep(C, DIMS, parity, oracle.COULOMB, oracle.STOCHASTIC, 1.0, 0.7, 5, parity)
        assert np.array_equal(C, B)
        assert n == 3
    finally:
        oracle.set_threads(1)


def test_update_links8_is_the_site_visit_of_the_sweep():
    U = gi.smooth_random_gauge(DIMS, 0.5, 16)
    nt, nx, ny, nz = DIMS
    flat = U.reshape(-1, 4, 3, 3)
    s = 2 + nx * (1 + ny * (3 + nz * 2))          # (x,y,z,t) = (2,1,3,2): parity 0
    c = {0: 2, 1: 2, 2: 1, 3: 3}                  # c[mu]
    stride = {0: nx * ny * nz, 1: 1, 2: nx, 3: nx * ny}
    back = [s - stride[mu] for mu in range(4)]    # no wrap needed at this site
    fwd = np.ascontiguousarray(flat[s].copy())
    bwd = np.ascontiguousarray(np.stack([flat[back[mu], mu] for mu in range(4)]))
    u = oracle.site_uniforms(77, 4, s)
    g = oracle.update_links8(fwd, bwd, oracle.LANDAU, oracle.STOCHASTIC, 1.0, 0.6, u)
    W = U.copy()
    oracle.sweep(W, DIMS, 0, oracle.LANDAU, oracle.STOCHASTIC, 1.0, 0.6, 77, 4)
    Wf = W.reshape(-1, 4, 3, 3)
    assert np.array_equal(Wf[s], fwd)
    for mu in range(4):
        assert np.array_equal(Wf[back[mu], mu], bwd[mu])
        assert np.allclose(fwd[mu], g @ flat[s, mu], atol=1e-15)                    # eq. 3, g(x+mu) = 1
        assert np.allclose(bwd[mu], flat[back[mu], mu] @ g.conj().T, atol=1e-15)    # eq. 3, g(x-mu) = 1
    assert c[0] == 2


# ------------------------------------------------------------------------- the fix loop

@pytest.mark.parametrize("seed", [0, 1, 2, 3, 4])
def test_config1_converges_to_1e12(seed):
    """BASELINE.json configs[0]: 4^4, eps = 0.3 smooth + Haar gauge, omega = 1.7, theta < 1e-12."""
    dims = (4, 4, 4, 4)
    U = gi.smooth_random_gauge(dims, 0.3, seed)
    U0 = U.copy()
    P0 = oracle.plaquette(U, dims)
    assert oracle.theta(U, dims) > 1e-2
    it, th, conv = oracle.fix_until(U, dims, oracle.LANDAU, oracle.OVERRELAX, 1.7, theta_target=1e-12,
                                    max_iter=2000, check_every=1)
    assert conv and th < 1e-12 and 20 < it < 400
    assert abs(oracle.theta(U, dims) - th) == 0.0
    assert abs(oracle.plaquette(U, dims) - P0) < 1e-12
    d_unit, d_det = oracle.unitarity_defect(U, dims)
    assert d_unit < 1e-12 and d_det < 1e-12
    assert oracle.functional(U, dims) > oracle.functional(U0, dims) + 0.3
    # the loop is exactly "parity 0 then parity 1, test theta": redo it by hand
    W = U0.copy()
    for k in range(it):
        oracle.sweep(W, dims, 0, oracle.LANDAU, oracle.OVERRELAX, 1.7)
        oracle.sweep(W, dims, 1, oracle.LANDAU, oracle.OVERRELAX, 1.7)
        assert (oracle.theta(W, dims) < 1e-12) == (k == it - 1)
    assert np.array_equal(W, U)


def test_coulomb_stochastic_converges_per_slice():
    """Reading A17 on a small replica of configs[4]: spatial K, per-slice theta_t, temporal links
    transformed too (plaquette incl. temporal planes invariant), slices decoupled."""
    dims = (6, 4, 4, 4)
    U = gi.smooth_random_gauge(dims, 0.6, 1)
    P0 = oracle.plaquette(U, dims)
    it, th, conv = oracle.fix_until(U, dims, oracle.COULOMB, oracle.STOCHASTIC, 1.0, 0.8, seed=2013,
                                    theta_target=1e-12, max_iter=5000, check_every=5)
    assert conv and th < 1e-12 and it % 5 == 0
    assert np.all(oracle.theta(U, dims, oracle.COULOMB) < 1e-12)
    assert abs(oracle.plaquette(U, dims) - P0) < 1e-12
    assert oracle.theta(U, dims, oracle.LANDAU) > 1e-6      # Coulomb-fixed is not Landau-fixed


def test_fix_loop_is_the_sequence_of_half_sweeps_with_consecutive_counters():
    """SURVEY 8(c) O5 / reading A10: iteration `it` of the fix loop is sweep(parity 0) with half-sweep counter
    first + 2 (it - 1), then sweep(parity 1) with first + 2 (it - 1) + 1 -- every half-sweep draws from its own
    Philox stream.  The loop (stochastic, so that the counters matter) must leave bitwise the field of that explicit
    sequence, and not the field of a sequence in which both parities of an iteration share a counter."""
    dims = (4, 4, 4, 6)
    U = gi.smooth_random_gauge(dims, 0.5, 17)
    A = U.copy()
    it, th, conv = oracle.fix_until(A, dims, oracle.COULOMB, oracle.STOCHASTIC, 1.0, 0.7, seed=99, first_counter=6,
                                    theta_target=0.0, max_iter=3, check_every=1)
    assert it == 3 and not conv
    B, C = U.copy(), U.copy()
    for k in range(3):
        for parity in (0, 1):
            oracle.sweep(B, dims, parity, oracle.COULOMB, oracle.STOCHASTIC, 1.0, 0.7, seed=99, half_sweep_counter=6 + 2 * k + parity)
            oracle.sweep(C, dims, parity, oracle.COULOMB, oracle.STOCHASTIC, 1.0, 0.7, seed=99, half_sweep_counter=6 + 2 * k)
    assert np.array_equal(A, B)
    assert not np.array_equal(B, C)
    assert th == np.max(oracle.theta(B, dims, oracle.COULOMB))


def test_coulomb_slices_are_decoupled():
    """Temporal links never enter K (A17): changing slice t' != t leaves slice t's spatial links'
    evolution unchanged."""
    dims = (4, 4, 4, 4)
    U = gi.smooth_random_gauge(dims, 0.5, 3)
    W = U.copy()
    W[3] = gi.hot_links((1, 4, 4, 4), 9)[0]           # replace everything stored on slice t = 3
    for k in range(3):
        for parity in (0, 1):
            oracle.sweep(U, dims, parity, oracle.COULOMB, oracle.OVERRELAX, 1.6)
            oracle.sweep(W, dims, parity, oracle.COULOMB, oracle.OVERRELAX, 1.6)
    assert np.array_equal(U[1, ..., 1:, :, :], W[1, ..., 1:, :, :])     # spatial links of slice 1
    assert not np.allclose(U[3], W[3])


# ----------------------------------------- the accumulated transformation (eq. 3)

def test_apply_transform_is_eq3_and_a_gauge_transformation():
    """oracle.apply_transform (C loops) against the input generator's independent numpy statement of
    eq. 3; identity and composition laws; the plaquette does not see it."""
    dims = (4, 6, 4, 8)
    U = gi.smooth_random_gauge(dims, 0.4, 3)
    G = gi.random_gauge(dims, 11)
    out = oracle.apply_transform(U, G, dims)
    assert np.abs(out - gi.gauge_transform(U, G)).max() < 1e-14
    assert np.array_equal(oracle.apply_transform(U, oracle.identity_transform(dims), dims), U)
    H = gi.random_gauge(dims, 12)
    HG = np.ascontiguousarray(np.einsum("...ab,...bc->...ac", H, G))
    assert np.abs(oracle.apply_transform(out, H, dims) - oracle.apply_transform(U, HG, dims)).max() < 1e-14
    assert abs(oracle.plaquette(out, dims) - oracle.plaquette(U, dims)) < 1e-14
    # a transposed or un-daggered neighbour matrix would break both
    x = (1, 2, 3, 4)          # (t, z, y, x)
    xp = (1, 2, 3, 5)         # x + x_hat
    assert np.abs(out[x][1] - G[x] @ U[x][1] @ G[xp].conj().T).max() < 1e-14


@pytest.mark.parametrize("gauge,algo", [(oracle.LANDAU, oracle.OVERRELAX), (oracle.COULOMB, oracle.STOCHASTIC)])
def test_accumulated_transformation_reproduces_the_swept_links(gauge, algo):
    """Gtot(x) <- g(x) Gtot(x): after any number of half-sweeps the links are
    Gtot(x) U0_mu(x) Gtot(x+mu)^dagger of the initial links (eq. 3), Gtot stays in SU(3), and the
    links are bitwise those of the plain sweep."""
    dims = (4, 4, 6, 4)
    U0 = gi.smooth_random_gauge(dims, 0.5, 21)
    U, Uplain = U0.copy(), U0.copy()
    G = oracle.identity_transform(dims)
    for it in range(3):
        for parity in (0, 1):
            kw = dict(gauge=gauge, algo=algo, omega=1.7, p=0.7, seed=5, half_sweep_counter=2 * it + parity)
            oracle.sweep_accumulate(U, G, dims, parity, **kw)
            oracle.sweep(Uplain, dims, parity, **kw)
            if it == 0 and parity == 0:
                # only the visited parity has moved away from the identity
                par = np.indices(G.shape[:4]).sum(axis=0) % 2
                assert np.all(G[par == 1] == np.eye(3))
                assert np.abs(G[par == 0] - np.eye(3)).max() > 1e-3
    assert np.array_equal(U, Uplain)
    assert np.abs(oracle.apply_transform(U0, G, dims) - U).max() < 1e-13
    GG = np.einsum("...ab,...cb->...ac", G, G.conj())
    assert np.abs(GG - np.eye(3)).max() < 1e-13
    assert np.abs(np.linalg.det(G) - 1).max() < 1e-13


# ------------------------------------------------- Coulomb gauge: frozen slices (reading A17b)

def test_masked_sweep_skips_exactly_the_frozen_slices():
    dims = (6, 4, 4, 4)
    U0 = gi.smooth_random_gauge(dims, 0.5, 8)
    kw = dict(gauge=oracle.COULOMB, algo=oracle.STOCHASTIC, p=0.6, seed=3, half_sweep_counter=4)
    A, B = U0.copy(), U0.copy()
    oracle.sweep_masked(A, dims, 0, [1] * 6, **kw)
    oracle.sweep(B, dims, 0, **kw)
    assert np.array_equal(A, B)                                  # all active = the plain sweep
    C = U0.copy()
    oracle.sweep_masked(C, dims, 0, [1, 0, 1, 1, 0, 1], **kw)
    oracle.sweep_masked(C, dims, 1, [1, 0, 1, 1, 0, 1], **dict(kw, half_sweep_counter=5))
    oracle.sweep(B, dims, 1, **dict(kw, half_sweep_counter=5))
    for t in (1, 4):                                             # frozen: spatial links untouched, theta_t unchanged
        assert np.array_equal(C[t][..., 1:, :, :], U0[t][..., 1:, :, :])
    th0, thC, thB = (oracle.theta(X, dims, oracle.COULOMB) for X in (U0, C, B))
    assert thC[1] == th0[1] and thC[4] == th0[4]
    for t in (0, 2, 3, 5):                                       # active slices evolve as if nothing were frozen
        assert np.array_equal(C[t][..., 1:, :, :], B[t][..., 1:, :, :])
        assert thC[t] == thB[t]
    # the temporal links leaving a frozen slice are still rotated by the active slice above it
    assert not np.array_equal(C[1][..., 0, :, :], U0[1][..., 0, :, :])
    assert abs(oracle.plaquette(C, dims) - oracle.plaquette(U0, dims)) < 1e-14


def test_fix_until_freeze_fixes_every_slice_as_the_unfrozen_run_does():
    """Each slice ends exactly where the unfrozen run had it at the iteration it was frozen (slices are
    decoupled); every theta_t < target; the run is still a gauge transformation."""
    dims = (6, 4, 4, 6)
    U0 = gi.smooth_random_gauge(dims, 0.4, 31)
    kw = dict(algo=oracle.OVERRELAX, omega=1.6)
    U = U0.copy()
    it, th, frozen_at, conv = oracle.fix_until_freeze(U, dims, theta_target=1e-12, max_iter=3000, check_every=1, **kw)
    assert conv and np.all(th < 1e-12) and np.all(frozen_at > 0) and it == frozen_at.max()
    assert len(set(frozen_at.tolist())) > 1                      # the slices do converge at different times
    assert np.array_equal(th, oracle.theta(U, dims, oracle.COULOMB))
    assert abs(oracle.plaquette(U, dims) - oracle.plaquette(U0, dims)) < 1e-13
    W = U0.copy()
    for n in range(1, it + 1):
        for parity in (0, 1):
            oracle.sweep(W, dims, parity, gauge=oracle.COULOMB, half_sweep_counter=2 * (n - 1) + parity, **kw)
        for t in np.nonzero(frozen_at == n)[0]:
            assert np.array_equal(W[t][..., 1:, :, :], U[t][..., 1:, :, :])
    # and it stops no later than the unfrozen loop
    it_plain, _, conv_plain = oracle.fix_until(U0.copy(), dims, gauge=oracle.COULOMB, theta_target=1e-12, max_iter=3000,
                                               check_every=1, **kw)
    assert conv_plain and it == it_plain


def test_fix_loops_refuse_more_time_slices_than_their_per_slice_state_holds():
    """oracle_fix_until / oracle_fix_until_freeze keep theta_t / the active flags in arrays of 4096 entries (the
    library's own limit on N_t): a longer lattice is refused instead of overrunning them; 4096 itself still runs."""
    long = (4098, 2, 2, 2)
    U = gi.unit_links(long)
    with pytest.raises(ValueError):
        oracle.fix_until(U, long, oracle.COULOMB, max_iter=1)
    with pytest.raises(ValueError):
        oracle.fix_until_freeze(U, long, max_iter=1)
    ok = (4096, 2, 2, 2)
    it, th, conv = oracle.fix_until(gi.unit_links(ok), ok, oracle.COULOMB, max_iter=3)
    assert it == 1 and th == 0.0 and conv                  # unit links are fixed: the first evaluation stops
    it, th_t, frozen_at, conv = oracle.fix_until_freeze(gi.unit_links(ok), ok, max_iter=3)
    assert it == 1 and conv and (frozen_at == 1).all() and (th_t == 0.0).all()
