"""Pins of the fp64 oracle against what the paper and the mathematics fix (CPU only).

Each test names the PAPER.md passage (P:Lnnn) or DESIGN.md reading (R-n) it pins.
Nothing here touches the CUDA path.
"""
import math
import os

import numpy as np
import pytest
from scipy import special, stats

from oracle import jump_oracle as jo
from paper_2412_15073_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")
KB, KCAL, COUL = 1.987204259e-3, 418.4, 332.063713


# ---------------------------------------------------------------- random numbers (R-15)
def test_philox_known_answers():
    for line in open(os.path.join(GOLD, "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        h = [int(t, 16) for t in line.split()]
        assert jo.philox(h[0:4], h[4:6]) == h[6:10]


def test_uniform_is_exact_in_fp32_and_open_interval():
    rng = np.random.default_rng(1)
    for w in list(rng.integers(0, 2 ** 32, size=2000)) + [0, 2 ** 32 - 1, 255, 256]:
        u = jo.u01(w)
        assert 0.0 < u < 1.0
        assert float(np.float32(u)) == u
    assert jo.u01(0) == 2.0 ** -24 and jo.u01(2 ** 32 - 1) == 1.0 - 2.0 ** -24


def test_philox_stream_moments():
    w = np.array([jo.philox([i, 3, 1, 0], [42, 0]) for i in range(20000)], dtype=np.uint64).ravel()
    u = ((w >> 9).astype(np.float64) + 0.5) / 2 ** 23
    assert abs(u.mean() - 0.5) < 4 * math.sqrt(1 / 12 / u.size)
    assert stats.kstest(u, "uniform").pvalue > 1e-3


# ---------------------------------------------------------------- chi and the split (R-3)
def test_chi_end_conditions_and_derivative():
    rc, h = 6.0, 0.5
    assert jo.chi(rc - h, rc, h) == (1.0, 0.0)
    assert jo.chi(rc, rc, h) == (0.0, 0.0)
    assert jo.chi(3.0, rc, h) == (1.0, 0.0) and jo.chi(7.0, rc, h) == (0.0, 0.0)
    d = 1e-6
    for r in np.linspace(rc - h + 0.01, rc - 0.01, 23):
        fd = (jo.chi(r + d, rc, h)[0] - jo.chi(r - d, rc, h)[0]) / (2 * d)
        assert abs(fd - jo.chi(r, rc, h)[1]) < 1e-8
        assert 0.0 < jo.chi(r, rc, h)[0] < 1.0
    # C^2 at both ends: chi' and chi'' vanish
    for r0, s in ((rc - h, +1), (rc, -1)):
        d1 = jo.chi(r0 + s * 1e-4, rc, h)[1]
        assert abs(d1) < 1e-5 * 30 / h
        for dd in (1e-4, 1e-5):      # chi'' = O(distance to the end): 60 u / h^2
            d2 = (jo.chi(r0 + s * 2 * dd, rc, h)[1] - jo.chi(r0 + s * dd, rc, h)[1]) / dd
            assert abs(d2) < 1.2 * 60 * (1.5 * dd / h) / h ** 2


def test_short_plus_long_is_unsplit():
    rc, h, rl, alpha = 5.0, 0.5, 9.0, 0.42
    for r in np.linspace(1.0, 8.99, 400):
        for (u, du) in (jo.u_coul(r, -0.3 * COUL, alpha), jo.u_lj(r, 3.15, 0.15)):
            s = jo.weighted_du(1, r, rc, h, rl, u, du) + jo.weighted_du(2, r, rc, h, rl, u, du)
            assert abs(s - jo.weighted_du(3, r, rc, h, rl, u, du)) <= 1e-13 * max(1.0, abs(du))
            assert abs(s - du) <= 1e-13 * max(1.0, abs(du))
            e = jo.weighted_u(1, r, rc, h, rl, u) + jo.weighted_u(2, r, rc, h, rl, u)
            assert abs(e - u) <= 1e-13 * max(1.0, abs(u))
    assert jo.weighted_du(3, 9.0, rc, h, rl, 1.0, 1.0) == 0.0      # neglected beyond r_long
    assert jo.weighted_du(1, 5.2, rc, h, rl, 1.0, 1.0) == 0.0      # short part vanishes beyond r_c
    assert jo.weighted_du(2, 4.4, rc, h, rl, 1.0, 1.0) == 0.0      # long part vanishes below r_c - h


def test_pair_potentials_closed_forms():
    alpha = 0.3167
    for r in (1.7, 3.3, 6.1, 11.0):
        u, du = jo.u_coul(r, 2.5, alpha)
        assert abs(u - 2.5 * special.erfc(alpha * r) / r) < 1e-15 * abs(u) + 1e-18
        d = 1e-6
        fd = (jo.u_coul(r + d, 2.5, alpha)[0] - jo.u_coul(r - d, 2.5, alpha)[0]) / (2 * d)
        assert abs(fd - du) < 1e-8 * max(abs(du), 1e-3)
        u, du = jo.u_lj(r, 3.1507, 0.1521)
        fd = (jo.u_lj(r + d, 3.1507, 0.1521)[0] - jo.u_lj(r - d, 3.1507, 0.1521)[0]) / (2 * d)
        assert abs(fd - du) < 1e-7 * max(abs(du), 1e-3)
    rmin = 2 ** (1 / 6) * 3.1507
    u, du = jo.u_lj(rmin, 3.1507, 0.1521)                         # textbook LJ: minimum -eps at 2^(1/6) sigma
    assert abs(u + 0.1521) < 1e-14 and abs(du) < 1e-13
    assert abs(jo.u_lj(3.1507, 3.1507, 0.1521)[0]) < 1e-15        # zero at sigma
    assert abs(jo.u_coul(2.0, COUL, 0.0)[0] - COUL / 2.0) < 1e-12  # alpha = 0: bare Coulomb


# ---------------------------------------------------------------- Theta (R-5)
def test_theta_values_and_identities():
    for line in open(os.path.join(GOLD, "theta_values.txt")):
        if line.startswith("#") or not line.strip():
            continue
        eta, val = map(float, line.split())
        assert abs(jo.theta(eta) - val) < 2e-10
    for eta in np.linspace(-6, 6, 49):
        assert abs(jo.theta(eta) - jo.theta(-eta) - eta) < 1e-14
        assert jo.theta(eta) <= max(eta, 0.0) + 1 / math.sqrt(2 * math.pi) + 1e-15   # bound behind P:L374
        d = 1e-5
        assert abs((jo.theta(eta + d) - jo.theta(eta - d)) / (2 * d) - stats.norm.cdf(eta)) < 1e-9
    g = np.random.default_rng(5).normal(size=2_000_000)
    for eta in (-1.5, 0.3, 2.0):
        mc = np.maximum(eta + g, 0).mean()
        assert abs(mc - jo.theta(eta)) < 5 * np.maximum(eta + g, 0).std() / math.sqrt(g.size)


# ---------------------------------------------------------------- G~ sampler (R-6)
def _gt_cdf(y, eta):
    y = np.maximum(y, -eta)
    num = eta * math.sqrt(2 * math.pi) * (stats.norm.cdf(y) - stats.norm.cdf(-eta)) + math.exp(-eta * eta / 2) - np.exp(-y * y / 2)
    return num / (math.sqrt(2 * math.pi) * jo.theta(eta))


def _gt_batch(eta, n, seed):
    import ctypes as C
    out = np.empty(n)
    L = jo.lib()
    L.orc_gtilde_batch.restype = C.c_int64
    L.orc_gtilde_batch.argtypes = [C.c_double, C.c_uint64, C.c_int, C.POINTER(C.c_double)]
    att = L.orc_gtilde_batch(float(eta), int(seed), n, out.ctypes.data_as(C.POINTER(C.c_double)))
    return out, att


@pytest.mark.parametrize("eta", [-6.0, -3.0, -2.5, -1.7, -1.0, -0.4, 0.0, 0.6, 2.0, 5.0])
def test_gtilde_distribution(eta):
    n = 200_000
    y, att = _gt_batch(eta, n, seed=11)
    assert (y > -eta).all()
    assert stats.kstest(y, lambda t: _gt_cdf(t, eta)).pvalue > 1e-3
    mean = stats.norm.cdf(eta) / jo.theta(eta)                     # E[G~] = Phi(eta)/Theta(eta)
    assert abs(y.mean() - mean) < 5 * y.std() / math.sqrt(n)
    rate = n / att
    lo = {-6.0: 0.9, -3.0: 0.7, -2.5: 0.45, -1.7: 0.45, -1.0: 0.33, -0.4: 0.5, 0.0: 0.999, 0.6: 0.75, 2.0: 0.75, 5.0: 0.75}[eta]
    assert rate >= lo                                              # acceptance-rate table of R-6


def test_gtilde_mean_golden():
    # E[G~] = Phi(eta)/Theta(eta): 1.2533 at 0, 0.4866 at 2, 3.5323 at -3
    for eta, val in ((0.0, 1.2533), (2.0, 0.4866), (-3.0, 3.5323)):
        y, _ = _gt_batch(eta, 400_000, seed=3)
        assert abs(y.mean() - val) < 6e-3


# ---------------------------------------------------------------- mechanism (6),(7): invariance of mu
def test_rate_and_kick_leave_gaussian_invariant():
    """(1/eps) E_u[Theta(eps u) E(f(u') - f(u))] = -E_u[f'(u)], u ~ N(0,1) the reduced velocity
    sqrt(beta m) v.n, u' given by the kick (7): stationarity of mu for one pair."""
    un, uw = np.polynomial.hermite_e.hermegauss(120)
    uw = uw / math.sqrt(2 * math.pi)
    yg = np.linspace(-14, 14, 56001)
    dy = yg[1] - yg[0]
    tests = [(np.sin, np.cos), (lambda t: t ** 3, lambda t: 3 * t ** 2),
             (lambda t: np.exp(-(t - 0.7) ** 2), lambda t: -2 * (t - 0.7) * np.exp(-(t - 0.7) ** 2))]
    for eps in (0.05, 0.3, 1.0, 3.0):
        for f, df in tests:
            lhs = 0.0
            for u, w in zip(un, uw):
                eta = eps * u
                if jo.theta(eta) < 1e-250:                             # weight x rate < 1e-250: no contribution
                    continue
                rate = jo.jump_rate(eps, 1.0, 1.0, 1.0, u)             # beta = m = g = 1
                assert abs(rate - jo.theta(eta) / eps) < 1e-14
                dens = np.maximum(eta + yg, 0) * np.exp(-yg * yg / 2) / (jo.theta(eta) * math.sqrt(2 * math.pi))
                # kick through the oracle's own routine, in 1-D: v = (u,0,0), n = (1,0,0), sbm = 1
                u1 = jo.jump_kick(eps, 1.0, [1, 0, 0], 0.0, [u, 0, 0])[0]      # gt = 0
                slope = jo.jump_kick(eps, 1.0, [1, 0, 0], 1.0, [u, 0, 0])[0] - u1
                up = u1 + slope * yg
                lhs += w * rate * (np.sum(dens * (f(up) - f(u))) * dy)
            rhs = -np.sum(uw * df(un))
            assert abs(lhs - rhs) < 2e-6 * max(1.0, abs(rhs)), (eps, lhs, rhs)


def test_eps_infinity_is_bps():
    # eps = inf is the BPS (4),(5)
    rng = np.random.default_rng(2)
    for _ in range(20):
        v = rng.normal(size=3) * 5
        n = rng.normal(size=3); n /= np.linalg.norm(n)
        g, beta, sbm = 0.37, 1.68, 0.25
        vn = float(v @ n)
        assert abs(jo.jump_rate(math.inf, beta, sbm, g, vn) - beta * g * max(vn, 0)) < 1e-15
        v2 = jo.jump_kick(math.inf, sbm, n, 123.0, v)
        assert np.allclose(v2, v - 2 * vn * n, atol=1e-14)
        assert abs(np.linalg.norm(v2) - np.linalg.norm(v)) < 1e-13
        # large finite eps approaches it
        big = 1e7
        assert abs(jo.jump_rate(big, beta, sbm, g, vn) - beta * g * max(vn, 0)) < 1e-5
        assert np.allclose(jo.jump_kick(big, sbm, n, 0.8, v), v - 2 * vn * n, atol=1e-5)


# ---------------------------------------------------------------- forces
@pytest.fixture(scope="module")
def cfg0():
    sysd, run = wl.make_config(0)
    return sysd, run


def _numpy_reference_forces(sysd, run, wC, wLJ):
    """Independent O(N^2) numpy restatement of grad U (R-2, R-3) for the pin."""
    x = sysd["pos"]; q = sysd["charge"]; sig = sysd["lj_sigma"]; eps = sysd["lj_eps"]
    n = x.shape[0]; L = sysd["box"]
    rc, h, rl = run["r_short"], run["r_switch"], run["r_long"]
    alpha = 3.8 / rl
    d = x[:, None, :] - x[None, :, :]
    d -= L * np.round(d / L)
    r = np.sqrt((d ** 2).sum(-1))
    mask = ~np.eye(n, dtype=bool)
    for i in range(n):
        mask[i, sysd["excl_idx"][sysd["excl_ptr"][i]:sysd["excl_ptr"][i + 1]]] = False
    mask &= r < rl
    r = np.where(mask, r, 1.0)
    u = np.clip((r - (rc - h)) / h, 0, 1)
    chi = 1 - 10 * u ** 3 + 15 * u ** 4 - 6 * u ** 5
    dchi = -30 * u ** 2 * (1 - u) ** 2 / h

    def weight(mode, U, dU):
        if mode == "short":
            return chi * dU + dchi * U
        if mode == "long":
            return (1 - chi) * dU - dchi * U
        return dU

    qq = COUL * q[:, None] * q[None, :]
    uC = qq * special.erfc(alpha * r) / r
    duC = -qq * (special.erfc(alpha * r) / r ** 2 + 2 * alpha / math.sqrt(math.pi) * np.exp(-(alpha * r) ** 2) / r)
    s = np.sqrt(sig[:, None] * sig[None, :]); e = np.sqrt(eps[:, None] * eps[None, :])
    uL = 4 * e * ((s / r) ** 12 - (s / r) ** 6)
    duL = 4 * e * (-12 * (s / r) ** 12 + 6 * (s / r) ** 6) / r
    fr = (weight(wC, uC, duC) + weight(wLJ, uL, duL)) * mask
    return (fr[:, :, None] * d / r[:, :, None]).sum(1)


def test_pair_forces_against_numpy_brute_force(cfg0):
    sysd, run = cfg0
    o = jo.Oracle(sysd, **run)
    for which, modes in ((4, ("short", "short")), (2, ("long", "long"))):
        ref = _numpy_reference_forces(sysd, run, *modes)
        got = o.forces(which)
        scale = np.sqrt((ref ** 2).sum(1).mean())
        assert np.abs(got - ref).max() < 1e-11 * scale
        assert np.abs(o.forces(which, brute=True) - got).max() < 1e-11 * scale
    full = o.forces(1) - o.forces(3)
    ref = _numpy_reference_forces(sysd, run, "full", "full")
    assert np.abs(full - ref).max() < 1e-10 * np.sqrt((ref ** 2).sum(1).mean())
    # F0 + long = full, Newton's third law
    assert np.abs(o.forces(0) + o.forces(2) - o.forces(1)).max() < 1e-11
    for w in (0, 1, 2, 3):
        assert np.abs(o.forces(w).sum(0)).max() < 1e-10


def test_forces_are_gradients_finite_difference(cfg0):
    sysd, run = cfg0
    o = jo.Oracle(sysd, **run)
    x0 = o.pos
    d = 1e-5
    rng = np.random.default_rng(0)
    for which in (0, 1, 2, 3):
        g = o.forces(which)
        for i in rng.choice(o.n, size=3, replace=False):
            for k in range(3):
                xp = x0.copy(); xp[i, k] += d
                xm = x0.copy(); xm[i, k] -= d
                o.set_state(xp, rebuild=False); ep = o.potential(which)
                o.set_state(xm, rebuild=False); em = o.potential(which)
                fd = (ep - em) / (2 * d)
                assert abs(fd - g[i, k]) < 2e-6 * max(1.0, abs(g[i, k])), (which, i, k, fd, g[i, k])
        o.set_state(x0, rebuild=False)


def test_bonded_zero_at_equilibrium_geometry():
    sysd, run = wl.make_config(0)
    o = jo.Oracle(sysd, **run)
    assert np.abs(o.forces(3)).max() < 3e-3      # generator places molecules at (r0, theta0), fp32-rounded
    assert abs(o.potential(3)) < 1e-6


def test_neighbor_search_matches_brute_force(cfg0):
    sysd, run = cfg0
    o = jo.Oracle(sysd, **run)
    for (lo, hi, lj) in ((0.0, 5.0, False), (3.5, 6.0, False), (6.0, 10.0, False), (3.5, 10.0, True)):
        p1, i1 = o.neighbors(lo, hi, lj, brute=False)
        p2, i2 = o.neighbors(lo, hi, lj, brute=True)
        assert np.array_equal(p1, p2) and np.array_equal(i1, i2)


def _contract_keys(x, box, edge):
    ng = np.maximum(1, np.floor(np.broadcast_to(box, (3,)) / edge).astype(int))
    cell = np.minimum(np.floor(x * (ng / box)).astype(int), ng - 1)
    return ng, cell, (cell[:, 2] * ng[1] + cell[:, 1]) * ng[0] + cell[:, 0]


def test_ring_rows_contract(cfg0):
    """R-10 (list_policy 0): M = [rc-h-s, rM), L = [rM, rlong+s), V = LJ pairs of the shell; ascending (cell key, index)."""
    sysd, run = cfg0
    o = jo.Oracle(sysd, **dict(run, list_policy=0))
    x = sysd["pos"]; L = sysd["box"]; n = o.n
    rc, h, s, rM, rl = run["r_short"], run["r_switch"], run["skin"], run["r_mid"], run["r_long"]
    _, _, key = _contract_keys(x, L, (rl + s) / 4)
    d = x[:, None, :] - x[None, :, :]
    d -= L * np.round(d / L)
    r = np.sqrt((d ** 2).sum(-1))
    nM, nL, nV = o.row_counts()
    for i in (0, 1, 2, 100, 331, 647):
        excl = set(sysd["excl_idx"][sysd["excl_ptr"][i]:sysd["excl_ptr"][i + 1]].tolist()) | {i}
        for which, lo_, hi_ in ((0, rc - h - s, rM), (1, rM, rl + s), (2, rc - h - s, rl + s)):
            want = [j for j in range(n) if j not in excl and lo_ <= r[i, j] < hi_
                    and (which != 2 or sysd["lj_eps"][i] * sysd["lj_eps"][j] > 0)]
            want.sort(key=lambda j: (key[j], j))
            got = o.row(which, i).tolist()
            assert got == want
    # symmetry: j in row(i) <=> i in row(j)
    i = 5
    for j in o.row(1, i):
        assert i in o.row(1, int(j))
    assert nV[1::3].max() == 0 and nV[::3].min() > 0     # LJ rows on oxygens only


@pytest.mark.parametrize("case", ["cfg0", "wide", "ortho"])
def test_rows_and_cell_universe_contract(cfg0, case):
    """R-10c (list_policy 1, the contract of the CUDA path): row A = [rc-h-s_ij, rA+s_ij), row B = [rA-s_ij, rM+s_ij) by
    build-time distance with the mass-weighted skin s_ij = (s/2)(w_i + w_j), w = m^-1/2 / mean(m^-1/2), excluded pairs
    never listed, ascending (cell key, index); ring 3 draws from the cell universe of the
    atom's home cell: the atoms of every contract cell within reach r_long + s of the home cell by the rule typed out
    below (an independent restatement), ascending (cell key, index), the atom itself and its excluded partners
    included.  And the property the thinning needs: every pair closer than r_long + s is in the universe."""
    sysd, run = cfg0
    if case == "wide":       # a box several stencils wide: the universe is a proper subset of the box
        sysd = wl.small_water(7, seed=4)                 # 1029 atoms, 31.3 A
        run = dict(run, r_short=4.0, r_long=5.5, r_mid=5.0, r_mid_in=4.25, skin=0.5, cell_edge=2.0)
    if case == "ortho":
        sysd = dict(wl.small_water(5, seed=13), box=np.array([16.0, 18.5, 21.0]))
        run = dict(run, r_short=4.0, r_long=7.5, r_mid=5.5, r_mid_in=4.5)
    o = jo.Oracle(sysd, **dict(run, list_policy=1))
    x = np.mod(sysd["pos"], sysd["box"]); n = o.n
    box = np.broadcast_to(np.asarray(sysd["box"], float), (3,))
    rc, h, s, rM, rl = run["r_short"], run["r_switch"], run["skin"], run["r_mid"], run["r_long"]
    rA = run.get("r_mid_in") or rc + 0.25
    w = 1.0 / np.sqrt(sysd["mass"]); w = w / w.mean()
    edge = run.get("cell_edge", 0.0) or (rl + s * w.max()) / 4
    ng, cell, key = _contract_keys(x, box, edge)
    d = x[:, None, :] - x[None, :, :]
    d -= box * np.round(d / box)
    r = np.sqrt((d ** 2).sum(-1))
    nA, nB, nU = o.row_counts()
    cw = box / ng
    reach = rl + s * w.max()
    R = np.ceil(reach / cw).astype(int)

    def cyc(a, b, m):
        o_ = (a - b) % m
        return min(o_, m - o_)

    def in_universe(ci, cj):
        a, b, e = cyc(cj[2], ci[2], ng[2]), cyc(cj[1], ci[1], ng[1]), cyc(cj[0], ci[0], ng[0])
        if a > R[2] or b > R[1]:
            return False
        rem = reach ** 2 - (max(a - 1, 0) * cw[2]) ** 2 - (max(b - 1, 0) * cw[1]) ** 2
        return rem > 0 and e <= min(R[0], int(math.floor(math.sqrt(rem) / cw[0])) + 1)

    for i in (0, 1, 2, 100, 331, n - 1):
        excl = set(sysd["excl_idx"][sysd["excl_ptr"][i]:sysd["excl_ptr"][i + 1]].tolist()) | {i}
        sij = 0.5 * s * (w[i] + w)
        for which, lo_, hi_ in ((0, rc - h, rA), (1, rA, rM)):
            want = [j for j in range(n) if j not in excl and max(lo_ - sij[j], 0.0) <= r[i, j] < hi_ + sij[j]]
            want.sort(key=lambda j: (key[j], j))
            assert o.row(which, i).tolist() == want
        want = [j for j in range(n) if in_universe(cell[i], cell[j])]
        want.sort(key=lambda j: (key[j], j))
        got = o.row(2, i).tolist()
        assert got == want and len(got) == nU[i]
        assert set(np.nonzero(r[i] < reach)[0].tolist()) <= set(got)       # superset of everything within reach
    if case == "wide":
        assert nU.max() < n                                                 # a proper subset


@pytest.mark.parametrize("policy", [0, 1])
def test_list_policies_give_the_same_accepted_jumps(relaxed_small, policy):
    """R-10 and R-10c list the candidate pairs differently (rows by build-time distance / rings by current distance with
    the cell universe) and so propose differently, but thinning makes the ACCEPTED jumps of every pair the same Poisson
    process: accepted events per chain and the mean kick agree between the two policies (frozen x, many
    replicas of one half-step), for the Coulomb and the LJ mechanism.  Run for policy 1 against the reference policy 0."""
    if policy == 0:
        pytest.skip("reference arm")
    sysd, kw = _frozen(relaxed_small, flags=1 | 2 | 4, eps_jump=1.0, skin=0.5, nlist_every=10 ** 9)
    res = []
    R = 1200
    for pol in (0, 1):
        o = jo.Oracle(sysd, **dict(kw, list_policy=pol))
        v0 = o.vel
        dv = np.zeros_like(v0)
        accC = accJ = 0
        for rep in range(R):
            o.set_vel(v0)
            o.clear_events()
            o.jump_half(4e-3, with_accel=False, step=rep + 50000 * pol)
            ev = o.events()
            accC += int(((ev["accepted"] == 1) & (ev["stream"] == 1)).sum())
            accJ += int(((ev["accepted"] == 1) & (ev["stream"] == 2)).sum())
            dv += o.vel - v0
        st = o.stats()
        assert st["max_p"] <= 1.0 and st["max_g_over_L"] <= 1.0
        res.append((st["proposals"] / R, accC / R, accJ / R, dv / R))
    (p0, c0, j0, d0), (p1, c1, j1, d1) = res
    assert abs(c1 / c0 - 1.0) < 5 * math.sqrt(2 / (c0 * R)) and c0 * R > 3000
    assert abs(j1 / j0 - 1.0) < 5 * math.sqrt(2 / (j0 * R)) and j0 * R > 100
    o = jo.Oracle(sysd, **kw)
    pred = -4e-3 * KCAL * o.forces(2) / sysd["mass"][:, None]
    proj = [(d * pred).sum() / (pred * pred).sum() for d in (d0, d1)]
    assert abs(proj[0] - proj[1]) < 0.3 and min(proj) > 0.3


@pytest.mark.parametrize("policy", [0, 1])
def test_bounds_dominate_every_listed_pair(cfg0, policy):
    sysd, run = cfg0
    o = jo.Oracle(sysd, **dict(run, list_policy=policy))
    b = o.bounds()
    q = sysd["charge"]
    rng = np.random.default_rng(3)
    worst = 0.0
    x = sysd["pos"]; L = sysd["box"]
    rc, h = run["r_short"], run["r_switch"]
    edges = (rc - h, b["rA"], b["rM"], run["r_long"])
    for i in rng.choice(o.n, size=40, replace=False):
        if policy == 0:
            for which, G in ((0, b["GM"]), (1, b["GL"])):
                for j in o.row(which, int(i)):
                    g, _ = o.fij(0, int(i), int(j))
                    worst = max(worst, g / (abs(q[i]) * b["qmax"] * G))
            for j in o.row(2, int(i)):
                g, _ = o.fij(1, int(i), int(j))
                worst = max(worst, g / (4 * math.sqrt(sysd["lj_eps"][i] * b["eps_max"]) * b["GV"]))
            continue
        # R-10c: a candidate carries its force through the ring its CURRENT distance lies in
        for which, G, GV in ((0, b["GM"], b["GV"]), (1, b["GL"], b["GV2"]), (2, b["G3"], b["GV3"])):
            for j in o.row(which, int(i)):
                if j == i:
                    continue
                d = x[i] - x[j]; d -= L * np.round(d / L)
                r = math.sqrt((d * d).sum())
                if not (edges[which] <= r < edges[which + 1]):
                    continue
                g, _ = o.fij(0, int(i), int(j))
                worst = max(worst, g / (abs(q[i]) * b["qmax"] * G))
                if sysd["lj_eps"][i] * sysd["lj_eps"][j] > 0:
                    g, _ = o.fij(1, int(i), int(j))
                    worst = max(worst, g / (4 * math.sqrt(sysd["lj_eps"][i] * b["eps_max"]) * GV))
    assert 0.5 < worst <= 1.0
    # values quoted in SURVEY R-7 for the (5, 9, 3.8/9) shape
    assert abs(b["GM"] - 0.993) < 2e-3


def test_lj_bound_covers_a_range_of_sigma():
    """sup_lj sweeps sigma_ij over [sigma_min, sigma_max] (R-7; inside the switching zone (1-chi) u' and
    -chi' u have opposite signs, so the sup over sigma is not at an end of the range by construction).  Two LJ species
    with sigma 3.0 and 4.0 A and different eps, both policies: over every listed pair (each ring under R-10c) the long
    LJ gradient stays below the bound, and the bound is not slack (max g / L > 0.5)."""
    rng = np.random.default_rng(12)
    n, box = 600, 26.0
    side = 9
    sites = np.array([(i, j, k) for i in range(side) for j in range(side) for k in range(side)])[rng.permutation(side ** 3)[:n]]
    pos = (sites + 0.5) * (box / side) + rng.uniform(-0.5, 0.5, size=(n, 3))
    z = np.zeros(0)
    sp = rng.integers(0, 2, size=n)
    sysd = dict(n_atoms=n, box=box, pos=np.mod(pos, box), vel=np.zeros((n, 3)), mass=np.full(n, 12.0), charge=np.zeros(n),
                lj_sigma=np.where(sp == 0, 3.0, 4.0), lj_eps=np.where(sp == 0, 0.05, 0.2),
                bond_ij=np.zeros((0, 2), dtype=np.int32), bond_k=z, bond_r0=z,
                angle_ijk=np.zeros((0, 3), dtype=np.int32), angle_k=z, angle_t0=z,
                excl_ptr=np.zeros(n + 1, dtype=np.int32), excl_idx=np.zeros(0, dtype=np.int32))
    for policy in (0, 1):
        o = jo.Oracle(sysd, r_short=5.0, r_long=9.0, r_mid=7.0, r_mid_in=5.25, skin=1.0, flags=2, list_policy=policy)
        b = o.bounds()
        assert b["sig_min"] == 3.0 and b["sig_max"] == 4.0 and b["eps_max"] == pytest.approx(0.2)
        x = np.mod(sysd["pos"], box)
        edges = (4.5, b["rA"], b["rM"], 9.0)
        worst = [0.0, 0.0, 0.0]
        for i in range(0, n, 7):
            for which, GV in ((2, b["GV"]),) if policy == 0 else ((0, b["GV"]), (1, b["GV2"]), (2, b["GV3"])):
                for j in o.row(which, i):
                    if j == i:
                        continue
                    d = x[i] - x[j]; d -= box * np.round(d / box)
                    r = math.sqrt((d * d).sum())
                    if policy == 1 and not (edges[which] <= r < edges[which + 1]):
                        continue
                    g, _ = o.fij(1, i, int(j))
                    k = 0 if policy == 0 else which
                    worst[k] = max(worst[k], g / (4 * math.sqrt(sysd["lj_eps"][i] * b["eps_max"]) * GV))
        assert max(worst) <= 1.0, worst
        assert worst[0] > 0.5, worst
        if policy == 1:
            assert worst[1] > 0.3 and worst[2] > 0.3, worst


# ---------------------------------------------------------------- integrator pieces
def _ideal_gas(n=4000, seed=0):
    rng = np.random.default_rng(seed)
    mass = np.where(np.arange(n) % 2 == 0, 16.0, 1.0)
    z = np.zeros(0)
    return dict(n_atoms=n, box=30.0, pos=rng.uniform(0, 30, size=(n, 3)), vel=np.zeros((n, 3)), mass=mass,
                charge=np.zeros(n), lj_sigma=np.ones(n), lj_eps=np.zeros(n),
                bond_ij=np.zeros((0, 2), dtype=np.int32), bond_k=z, bond_r0=z,
                angle_ijk=np.zeros((0, 3), dtype=np.int32), angle_k=z, angle_t0=z,
                excl_ptr=np.zeros(n + 1, dtype=np.int32), excl_idx=np.zeros(0, dtype=np.int32))


def test_O_step_is_exact_OU():
    # stationary variance k_B T / m whatever the time step; gamma = 0 is the identity
    sysd = _ideal_gas()
    o = jo.Oracle(sysd, r_short=5.0, r_long=9.0, dt_fs=50.0, gamma_per_ps=20.0, flags=0, seed=9, nlist_every=1000)
    o.jump_step(20)
    v = o.vel
    kT = KB * 300 * KCAL
    for m in (16.0, 1.0):
        sel = sysd["mass"] == m
        var = (v[sel] ** 2).mean()
        assert abs(var / (kT / m) - 1) < 5 * math.sqrt(2 / (3 * sel.sum()))
    o2 = jo.Oracle(dict(sysd, vel=v), r_short=5.0, r_long=9.0, dt_fs=1.0, gamma_per_ps=0.0, flags=0, nlist_every=1000)
    o2.jump_step(3)
    assert np.array_equal(o2.vel, v)
    assert np.allclose(o2.pos_unwrapped, np.mod(sysd["pos"], 30.0) + 3e-3 * v, atol=1e-12)


@pytest.fixture(scope="module")
def relaxed_small():
    """192-atom water box relaxed for a short while so that forces are liquid-like."""
    sysd = wl.small_water(4, seed=21)
    run = dict(r_short=4.0, r_long=6.0, r_mid=5.0, skin=0.2, nlist_every=1, dt_fs=0.5, gamma_per_ps=20.0, seed=5)
    o = jo.Oracle(sysd, **run)
    o.baoab_step(600)
    sysd = dict(sysd, pos=o.pos, vel=o.vel)
    return sysd, run


def test_baoab_energy_conservation_and_reversibility(relaxed_small):
    sysd, run = relaxed_small
    drift = []
    for dt in (0.5, 0.25):
        o = jo.Oracle(sysd, **dict(run, dt_fs=dt, gamma_per_ps=0.0))
        e = []
        for _ in range(int(40 / dt)):
            o.baoab_step(1)
            e.append(o.kinetic() + o.potential(1))
        drift.append(np.std(e))
    assert drift[0] < 0.05 * 192 * KB * 300            # tiny compared with the thermal energy
    assert 2.5 < drift[0] / drift[1] < 6.0             # O(dt^2)
    o = jo.Oracle(sysd, **dict(run, gamma_per_ps=0.0))
    x0, v0 = o.pos_unwrapped, o.vel
    o.baoab_step(50)
    o.set_state(vel=-o.vel, rebuild=False)
    xu = o.pos_unwrapped
    o.baoab_step(50)
    dx = o.pos_unwrapped - xu + (xu - x0)             # unwrapped copy restarts at set_state: compare via wrapped
    d = o.pos - np.mod(x0, sysd["box"])
    d -= sysd["box"] * np.round(d / sysd["box"])
    assert np.abs(d).max() < 1e-9
    assert np.abs(o.vel + v0).max() < 1e-8


def test_degenerate_cases_reduce_to_baoab(relaxed_small):
    sysd, run = relaxed_small
    # no charges and no LJ: no event can be accepted, chains only accelerate -> identical to jumps switched off
    neutral = dict(sysd, charge=np.zeros_like(sysd["charge"]), lj_eps=np.zeros_like(sysd["lj_eps"]))
    a = jo.Oracle(neutral, **dict(run, flags=3))
    b = jo.Oracle(neutral, **dict(run, flags=0))
    a.jump_step(5); b.jump_step(5)
    assert np.array_equal(a.pos, b.pos) and np.array_equal(a.vel, b.vel)
    assert a.stats()["proposals"] == 0
    # RESPA with jumps off and no outer force == n_inner plain steps (R-12)
    c = jo.Oracle(sysd, **dict(run, flags=0, n_inner=4))
    d = jo.Oracle(sysd, **dict(run, flags=0))
    c.jump_respa_step(2); d.jump_step(8)
    assert np.array_equal(c.pos, d.pos) and np.array_equal(c.vel, d.vel)


# ---------------------------------------------------------------- thinning and Algorithm 4/5
def _frozen(relaxed_small, **over):
    sysd, run = relaxed_small
    kw = dict(run, flags=1 | 4, eps_jump=0.3, nlist_every=10 ** 9)
    kw.update(over)
    return sysd, kw


@pytest.mark.parametrize("mode", [0, 1])
def test_event_log_invariants(relaxed_small, mode):
    sysd, kw = _frozen(relaxed_small, flags=1 | 2 | 4, eps_jump=1.0, eps_mode=mode)
    o = jo.Oracle(sysd, **kw)
    o.jump_step(3)
    ev = o.events()
    st = o.stats()
    assert st["max_p"] <= 1.0 and st["max_g_over_L"] <= 1.0     # thinning validity
    prop = ev[ev["ring"] >= 0]
    assert len(prop) == st["proposals"] and (ev["ring"] < 0).sum() == st["expiries"]
    assert np.array_equal(prop["accepted"] == 1, prop["U"] <= prop["p"])
    assert (prop["p"] >= 0).all() and (prop["p"] <= 1).all()
    # every chain ends with exactly one expiry, events of a chain fit in the half step
    H = 0.5 * kw["dt_fs"] * 1e-3
    keys = ev["step"].astype(np.int64) * 100000 * 16 + ev["stream"] * 100000 + ev["atom"]
    for kk in np.unique(keys)[:200]:
        ch = ev[keys == kk]
        assert (ch["ring"] < 0).sum() == 1 and ch["ring"][-1] < 0
        assert ch["T"][:-1].sum() <= H
        assert list(ch["iter"]) == list(range(len(ch)))
    # LJ chains only on oxygens (eps_i > 0), Coulomb chains on every atom
    assert (ev[ev["stream"] == 2]["atom"] % 3 == 0).all()
    assert set(np.unique(ev[ev["stream"] == 1]["atom"])) == set(range(o.n))
    # BPS reflections keep |v|: covered by test_eps_infinity_is_bps; partners come from the rows
    e0 = prop[(prop["stream"] == 1) & (prop["step"] == 0)][0]
    assert e0["j"] in o.row(int(e0["ring"]), int(e0["atom"]))


def _two_atoms(d=5.0, q=0.5):
    z = np.zeros(0)
    return dict(n_atoms=2, box=24.0, pos=np.array([[5.0, 5.0, 5.0], [5.0 + d, 5.0, 5.0]]), vel=np.zeros((2, 3)),
                mass=np.array([16.0, 1.0]), charge=np.array([q, -q]), lj_sigma=np.ones(2), lj_eps=np.zeros(2),
                bond_ij=np.zeros((0, 2), dtype=np.int32), bond_k=z, bond_r0=z,
                angle_ijk=np.zeros((0, 3), dtype=np.int32), angle_k=z, angle_t0=z,
                excl_ptr=np.zeros(3, dtype=np.int32), excl_idx=np.zeros(0, dtype=np.int32))


@pytest.mark.parametrize("eps,mode", [(0.3, 0), (2.0, 0), (15.0, 1)])
def test_mean_drift_of_jump_process_is_minus_F_over_m(eps, mode):
    """Averaged over Maxwellian velocities, rate (6) x mean kick (7) (E[G~] = Phi/Theta) gives exactly
    dE[v]/dt = -M^-1 F_ij for every eps -- the drift of the Hamiltonian flow the process replaces
    (P:L100-104).  Pins the sign convention R-4 and every factor of (6), (7).
    mode 1: adaptive eps(x) = eps0 |F_ij(x)| (R-19) -- at frozen x that is the constant eps0 g, so
    the same identity pins its rate, its bound (a p whose denominator were not the bound the clock runs on would
    change the effective rate) and its kernel."""
    sysd = _two_atoms()
    o = jo.Oracle(sysd, r_short=4.0, r_long=8.0, r_mid=6.0, skin=0.5, flags=1, eps_jump=eps, eps_mode=mode,
                  nlist_every=10 ** 9, seed=77)
    F = o.forces(2)
    assert np.abs(F[:, 0]).min() > 1e-3 and np.abs(F[:, 1:]).max() < 1e-12
    kT = KB * 300
    sbm = np.sqrt(sysd["mass"] / (kT * KCAL))
    if mode == 1:
        eps = eps * abs(F[0, 0])                              # the effective epsilon of the one pair (same |F| on both atoms)
        assert 0.2 < eps < 5.0
    rate0 = max(jo.jump_rate(eps, 1 / kT, sbm[i], abs(F[i, 0]), 0.0) for i in range(2))
    # mean rate over Maxwellian v is sqrt(1+eps^2) x the v = 0 rate; keep second events (bias) rare
    H = 0.02 / (rate0 * math.sqrt(1 + eps * eps))
    rng = np.random.default_rng(8)
    R = 300_000
    acc = np.zeros((2, 3))
    V = rng.normal(size=(R, 2, 3)) / sbm[None, :, None]
    for rep in range(R):
        o.set_vel(V[rep])
        o.jump_half(H, with_accel=False, step=rep)
        acc += o.vel - V[rep]
    mean = acc / R
    pred = -H * KCAL * F / sysd["mass"][:, None]
    assert o.stats()["accepts"] > 3000
    for i in range(2):
        assert abs(mean[i, 0] / pred[i, 0] - 1.0) < 0.06, (i, mean[i, 0], pred[i, 0])
        assert np.abs(mean[i, 1:]).max() < 0.05 * abs(pred[i, 0])


@pytest.mark.parametrize("mode", [0, 1])
def test_thinning_is_invariant_under_looser_bounds(relaxed_small, mode):
    # doubling every L doubles proposals and leaves the accepted-jump statistics unchanged; with the
    # adaptive eps (mode 1, R-19) only the beta L B_v part of the bound doubles, the accepted jumps still do not move
    sysd, kw = _frozen(relaxed_small, flags=1 | 2, eps_jump=1.0 if mode == 0 else 0.5, eps_mode=mode)
    res = []
    R = 1500
    for f in (1.0, 2.0):
        o = jo.Oracle(sysd, **kw)
        o.scale_bounds(f)
        v0 = o.vel
        dv = np.zeros_like(v0)
        for rep in range(R):
            o.set_vel(v0)
            o.jump_half(5e-4, with_accel=False, step=rep + 100000 * int(f))
            dv += o.vel - v0
        st = o.stats()
        res.append((st["proposals"] / R, st["accepts"] / R, dv / R))
    (p1, a1, d1), (p2, a2, d2) = res
    if mode == 0:
        assert abs(p2 / p1 - 2.0) < 5 * 2.0 * math.sqrt(1 / (p1 * R) + 1 / (p2 * R)) + 0.01
    else:
        assert 1.02 < p2 / p1 < 2.0
    assert abs(a2 / a1 - 1.0) < 5 * math.sqrt(2 / (a1 * R))
    o = jo.Oracle(sysd, **kw)
    pred = -5e-4 * KCAL * o.forces(2) / sysd["mass"][:, None]      # direction of the mean kick
    proj = [(d * pred).sum() / (pred * pred).sum() for d in (d1, d2)]
    assert abs(proj[0] - proj[1]) < 0.5 and min(proj) > 0.3   # noisy: the sharp check is the accept count


@pytest.mark.parametrize("policy", [0, 1])
def test_proposal_counts_are_poisson_for_bps(relaxed_small, policy):
    # Alg. 5 / P:L161: with |v| frozen the number of proposals of a chain is Poisson(beta |v| H sum_Y N_Y L_Y)
    # (one ring V under R-10, the three rings of R-10c)
    sysd, kw = _frozen(relaxed_small, flags=2 | 4, list_policy=policy)
    o = jo.Oracle(sysd, **kw)
    b = o.bounds()
    n0, n1, n2 = o.row_counts()
    v0 = o.vel
    H = 2e-3
    i = 0
    NG = n2[i] * b["GV"] if policy == 0 else n0[i] * b["GV"] + n1[i] * b["GV2"] + n2[i] * b["GV3"]
    lam = NG * (1 / (KB * 300)) * np.linalg.norm(v0[i]) * 4 * math.sqrt(sysd["lj_eps"][i] * b["eps_max"])
    counts = []
    for rep in range(400):
        o.clear_events()
        o.set_state(vel=v0, rebuild=False)
        o.jump_half(H, with_accel=False, step=rep)
        ev = o.events()
        counts.append(int(((ev["atom"] == i) & (ev["ring"] >= 4)).sum()))
    counts = np.array(counts)
    mu = lam * H
    assert abs(counts.mean() - mu) < 5 * math.sqrt(mu / len(counts))
    assert abs(counts.var() / mu - 1) < 0.3


def test_bound_held_between_accepted_jumps_is_algorithm_4(relaxed_small):
    """R-11: Algorithm 4 prints B_v and lambda-bar at every proposal; the oracle's default holds the bound
    evaluated at t = 0 / after an accepted jump until the next accepted jump ("re-evaluated after each jump").
    Both are valid bounds on [t, delta/2], so by P:L157 the accepted jumps have the same law and only the number of
    proposals differs: accepted events per chain and the mean velocity change agree between the two forms (frozen x,
    acceleration on, a half-step long enough for several events per chain), the held bound proposes a little more."""
    sysd, kw = _frozen(relaxed_small, flags=1, eps_jump=1.0)
    res = []
    R = 1500
    for every in (False, True):
        o = jo.Oracle(sysd, **kw)
        o.set_bound_mode(every)
        v0 = o.vel
        dv = np.zeros_like(v0)
        for rep in range(R):
            o.set_vel(v0)
            o.jump_half(5e-3, with_accel=True, step=rep + 200000 * int(every))
            dv += o.vel - v0
        st = o.stats()
        assert st["max_p"] <= 1.0
        res.append((st["proposals"] / R, st["accepts"] / R, dv / R))
    (p_held, a_held, d_held), (p_every, a_every, d_every) = res
    assert a_held * R > 5000
    assert abs(a_every / a_held - 1.0) < 5 * math.sqrt(2 / (a_held * R))
    assert 1.0 <= p_held / p_every < 1.5                      # looser bound: more proposals, never fewer
    assert np.abs(d_held - d_every).max() < 6 * np.abs(d_held).std() / math.sqrt(R) + 0.05 * np.abs(d_held).max()


def test_respa_proposals_per_time_independent_of_outer_step(relaxed_small):
    # the jump cost per unit simulated time does not depend on the level it sits in
    sysd, run = relaxed_small
    rates = []
    for n_inner in (2, 4):
        o = jo.Oracle(sysd, **dict(run, n_inner=n_inner, flags=3, dt_fs=0.5, nlist_every=4, skin=0.4))
        o.jump_respa_step(40 // n_inner)
        rates.append(o.stats()["proposals"] / (20 * 0.5))
    o = jo.Oracle(sysd, **dict(run, flags=3, dt_fs=0.5, nlist_every=4, skin=0.4))
    o.jump_step(40)
    rates.append(o.stats()["proposals"] / (20 * 0.5))
    assert abs(rates[0] / rates[1] - 1) < 0.1 and abs(rates[2] / rates[1] - 1) < 0.15


def test_jump_and_baoab_sample_the_same_measure(relaxed_small):
    """the hybrid jump process leaves mu invariant, so its long-run averages equal BAOAB's (which
    integrates the whole gradient of the same U).  192 atoms, 6 ps each after 1 ps of burn-in; kinetic temperature
    and potential energy per molecule with block-average error bars from four 1.5 ps blocks (the potential energy of
    water decorrelates over about 1 ps at gamma = 1 / ps: shorter blocks understate the error) (BASELINE.json north_star: "the hybrid process
    still samples mu").  A wrong rate, kick amplitude or sign heats or cools the system by tens of K within a ps
    (the Langevin thermostat acts on a 1 ps scale only)."""
    import observables as ob
    sysd, _ = relaxed_small
    run = dict(r_short=4.0, r_long=6.0, r_mid=5.0, skin=1.0, nlist_every=10, dt_fs=1.0, gamma_per_ps=1.0, eps_jump=1.0, flags=3)
    out = {}
    for name, seed in (("jump", 11), ("baoab", 12), ("adaptive", 13), ("bjaoajb", 14), ("combined", 15)):
        kw = dict(run, seed=seed)
        if name == "adaptive":                                 # eps(x) = eps0 |F_ij(x)| (R-19)
            kw.update(eps_mode=1, eps_jump=0.5)
        if name == "bjaoajb":                                  # B J A O A J B
            kw.update(flags=3 | jo.F_BJAOAJB)
        if name == "combined":                                 # one mechanism for Coulomb + LJ (R-22)
            kw.update(flags=3 | jo.F_COMBINED)
        o = jo.Oracle(sysd, **kw)
        step = o.baoab_step if name == "baoab" else o.jump_step
        step(1000)
        T, U = [], []
        for _ in range(600):
            step(10)
            T.append(o.temperature())
            U.append(o.potential(1) / 64.0)
        if name != "baoab":
            st = o.stats()
            assert st["accepts"] > 1000 and st["max_p"] <= 1.0 + 1e-9
        out[name] = (ob.block_mean_se(T, 4), ob.block_mean_se(U, 4))
        o.close()
    (Tj, Uj), (Tb, Ub) = out["jump"], out["baoab"]
    # The kinetic temperature read at the end of a step carries each splitting's own O(delta^2) bias (stiff O-H
    # bonds, omega delta = 0.7 at 1 fs): six 6-ps oracle runs of this box give 302.6 +- 2 K for JUMP and 291 +- 2 K for
    # BAOAB.  The slack is that 12 K offset; a wrong rate or kick shows up as tens of K.
    assert ob.agree(Tj, Tb, 4.0, slack=12.0), (Tj, Tb)       # K
    assert abs(Tj[0] - 300.0) < 20.0 and abs(Tb[0] - 300.0) < 20.0
    # the same bias in the mean potential energy: 0.09 - 0.1 kcal/mol per molecule in those runs (-1.61 against -1.70);
    # tests/test_gpu_longrun.py shows it falling fourfold at delta = 0.5 fs
    assert ob.agree(Uj, Ub, 4.0, slack=0.15), (Uj, Ub)       # kcal/mol per molecule
    for name in ("adaptive", "bjaoajb", "combined"):
        Ta, Ua = out[name]
        assert ob.agree(Ta, Tb, 4.0, slack=12.0) and abs(Ta[0] - 300.0) < 20.0, (name, Ta, Tb)
        assert ob.agree(Ua, Ub, 4.0, slack=0.15), (name, Ua, Ub)


@pytest.mark.parametrize("variant", ["accel", "jumps_only"])
def test_two_body_boltzmann_histogram(variant):
    """SURVEY C.6 "2-body toy"; invariance of mu.  One fixed charge (mass 1e8) and 24 light mobile charges that
    interact with it only (all mobile-mobile pairs are on the exclusion list): 24 copies of a two-body problem whose
    stationary law is known in closed form -- the distance r to the fixed charge has density ~ r^2 exp(-beta U(r)) on
    r <= box/2, U = u(r) - u(r_long) below r_long and 0 beyond (forces are truncated at r_long).  The whole
    C' machinery (clock, ring pick, candidate draw, rate (6), bound, acceptance, G~, kick (7), the drift of v under a
    before eta is formed) has to be right for the histogram of a long JUMP run to match it.
      accel:      Coulomb r_c = 5 A: short part in F0, rings [4.5, 7) by jumps; an LJ term (LJ jumps off, so it stays in
                  F0, R-13) accelerates the atoms everywhere in the rings (a != 0 while jumps happen);
      jumps_only: r_c = 1 A, no LJ: F0 = 0 wherever an atom ever is (a = 0), every force acts through jumps.
    Block averages over 20 blocks give the error bars; the laws without the jumped part are rejected by far."""
    rng = np.random.default_rng(1)
    box, nmob, q, al = 16.0, 24, 0.3, 0.25
    n = nmob + 1
    pos = np.zeros((n, 3)); pos[0] = [8.0, 8.0, 8.0]
    pos[1:] = rng.uniform(0, box, size=(nmob, 3))
    near = np.linalg.norm(pos[1:] - pos[0], axis=1) < 3.0
    pos[1:][near] += 4.0
    mass = np.r_[1e8, np.full(nmob, 1.0)]
    lj_eps, lj_sig = np.zeros(n), np.ones(n)
    if variant == "accel":
        lj_eps[:] = 1.0; lj_sig[:] = 3.5
    vel = rng.normal(size=(n, 3)) * np.sqrt(KB * 300 * KCAL / mass)[:, None]
    lists = [[]] + [[j for j in range(1, n) if j != i] for i in range(1, n)]
    ptr = np.zeros(n + 1, np.int32); ptr[1:] = np.cumsum([len(l) for l in lists])
    z = np.zeros(0)
    sysd = dict(n_atoms=n, box=box, pos=np.mod(pos, box), vel=vel, mass=mass, charge=np.full(n, q), lj_sigma=lj_sig,
                lj_eps=lj_eps, bond_ij=np.zeros((0, 2), np.int32), bond_k=z, bond_r0=z,
                angle_ijk=np.zeros((0, 3), np.int32), angle_k=z, angle_t0=z, excl_ptr=ptr,
                excl_idx=np.array([j for l in lists for j in l], np.int32))
    kw = dict(r_short=5.0, r_switch=0.5, r_mid_in=5.25, r_mid=6.0, r_long=7.0) if variant == "accel" else \
        dict(r_short=1.0, r_switch=0.5, r_mid_in=3.0, r_mid=5.0, r_long=7.0)
    o = jo.Oracle(sysd, ewald_alpha=al, dt_fs=2.0, gamma_per_ps=2.0, flags=1, eps_jump=1.0, skin=1.0, nlist_every=2, seed=1, **kw)
    o.jump_step(2000)
    nb, K, per = 11, 20, 4000
    edges = np.linspace(2.5, 8.0, nb + 1)
    H = np.zeros((K, nb))
    for k in range(K):
        for _ in range(per // 10):
            o.jump_step(10)
            d = o.pos[1:] - o.pos[0]
            d -= box * np.round(d / box)
            H[k] += np.histogram(np.linalg.norm(d, axis=1), bins=edges)[0]
    st = o.stats()
    assert st["max_p"] <= 1.0 and st["max_g_over_L"] <= 1.0 and st["accepts"] > 2000 and st["max_disp"] < 0.5
    beta = 1.0 / (KB * 300)

    def law(u_of_r):                               # bin probabilities of r^2 exp(-beta U), U shifted to 0 at r_long
        rr = np.linspace(2.5, 8.0, 110001)
        w = rr * rr * np.exp(-beta * np.where(rr < 7.0, u_of_r(rr) - u_of_r(7.0), 0.0))
        cdf = np.concatenate([[0.0], np.cumsum(0.5 * (w[1:] + w[:-1]) * np.diff(rr))])
        p = np.diff(np.interp(edges, rr, cdf))
        return p / p.sum()

    u_c = lambda r: 332.063713 * q * q * special.erfc(al * r) / r
    u_lj = lambda r: 4.0 * ((3.5 / r) ** 12 - (3.5 / r) ** 6) if variant == "accel" else 0.0 * r
    full = law(lambda r: u_c(r) + u_lj(r))
    P = H / H.sum(1, keepdims=True)
    m, se = P.mean(0), P.std(0, ddof=1) / math.sqrt(K)
    ok = full > 0.02                               # bins that are populated
    assert ok.sum() >= 7 and (se[ok] / full[ok]).max() < 0.06
    zs = (m[ok] - full[ok]) / se[ok]
    assert np.abs(zs).max() < 4.0, zs
    # the same run rejects the law without the part of U the jumps carry (their force replaced by nothing)
    def u_without_jumps(r):
        chi = np.array([jo.chi(x, kw["r_short"], 0.5)[0] for x in np.atleast_1d(r)])
        return chi * u_c(r) + u_lj(r)
    rr = np.linspace(2.5, 8.0, 2201)
    w = rr * rr * np.exp(-beta * (u_without_jumps(rr) - u_without_jumps(np.array([7.999]))[0]))
    cdf = np.concatenate([[0.0], np.cumsum(0.5 * (w[1:] + w[:-1]) * np.diff(rr))])
    alt = np.diff(np.interp(edges, rr, cdf)); alt /= alt.sum()
    assert (((m[ok] - alt[ok]) / se[ok]) ** 2).sum() > 150.0


def test_bjaoajb_scheme(relaxed_small):
    """B J A O A J B: with no jump mechanism it IS BAOAB with F0 (bit for bit the same as the C'
    scheme without jumps, whose event-free (C) is the same kick); with jumps the (J) parts run on a piecewise
    constant velocity: the chains of a step see a = 0, so every chain's first bound is beta S |v| + S lam0 and
    the events differ from the C'J'AOAJ'C' scheme's while the proposal rate stays the same to O(delta)."""
    sysd, run = relaxed_small
    kw = dict(run, dt_fs=1.0, gamma_per_ps=1.0, skin=1.0, nlist_every=10)
    a, b = jo.Oracle(sysd, **dict(kw, flags=jo.F_BJAOAJB)), jo.Oracle(sysd, **dict(kw, flags=0))
    a.jump_step(25); b.jump_step(25)
    assert np.array_equal(a.pos, b.pos) and np.array_equal(a.vel, b.vel) and a.stats()["proposals"] == 0
    a, b = jo.Oracle(sysd, **dict(kw, flags=3 | 4 | jo.F_BJAOAJB)), jo.Oracle(sysd, **dict(kw, flags=3 | 4))
    a.jump_step(20); b.jump_step(20)
    ea, eb = a.events(), b.events()
    assert set(np.unique(ea["stream"])) == {1, 2, 3, 4}
    assert len(ea) != len(eb) or not np.array_equal(ea["T"], eb["T"])
    ra, rb = a.stats()["proposals"], b.stats()["proposals"]
    assert abs(ra / rb - 1.0) < 0.05
    assert a.stats()["max_p"] <= 1.0 and np.abs(a.pos - b.pos).max() > 1e-6
    # one step by hand: B, J at frozen x with a = 0 (jump_half), A O A, J, B reproduce jump_step(1)
    c = jo.Oracle(sysd, **dict(kw, flags=3 | jo.F_BJAOAJB, gamma_per_ps=0.0))
    d = jo.Oracle(sysd, **dict(kw, flags=3, gamma_per_ps=0.0))
    c.jump_step(1)
    H = 0.5e-3
    f0 = d.forces(0)
    d.set_vel(d.vel - H * KCAL * f0 / sysd["mass"][:, None])
    d.jump_half(H, with_accel=False, step=0)                 # opening C'J' streams (1, 2) with a = 0
    x = d.pos + 2 * H * d.vel                                # A O A with gamma = 0
    assert np.abs((c.pos - x + 6.0) % sysd["box"] - 6.0).max() < 1e-12


def test_pair_histogram_lattice_and_ideal_gas():
    """NEXT-4 oracle pin: on a simple cubic lattice the neighbour shells are known in closed form (6 at a, 12 at
    a sqrt 2, 8 at a sqrt 3, 6 at 2a per site, each pair once); for uniform random points g(r) = 1."""
    n, a = 6, 2.0
    g = np.stack(np.meshgrid(*[np.arange(n)] * 3, indexing="ij"), -1).reshape(-1, 3) * a
    h = jo.pair_histogram(g, n * a, 4.1, 41)                      # bins of 0.1
    N = n ** 3
    expect = {20: 6 * N // 2, 28: 12 * N // 2, 34: 8 * N // 2, 40: 6 * N // 2}      # floor(r / 0.1)
    for b in range(41):
        assert h[b] == expect.get(b, 0), (b, h[b])
    rng = np.random.default_rng(3)
    box, M = 20.0, 3000
    h = jo.pair_histogram(rng.uniform(0, box, size=(M, 3)), box, 8.0, 16)
    edges = np.linspace(0, 8.0, 17)
    ideal = 0.5 * M * (M - 1) / box ** 3 * 4 / 3 * np.pi * (edges[1:] ** 3 - edges[:-1] ** 3)
    assert np.abs(h[2:] / ideal[2:] - 1).max() < 5 / np.sqrt(ideal[2:].min())


# ---------------------------------------------------------------- NEXT-2: reciprocal Ewald sum as F_{0,1}, JUMP-RESPA1 (R-21)
def _rock_salt(cells=2, d=1.0):
    """(2 cells)^3 rock-salt lattice of unit charges, nearest-neighbour distance d."""
    m = 2 * cells
    g = np.array([(i, j, k) for i in range(m) for j in range(m) for k in range(m)])
    n = len(g)
    z = np.zeros(0)
    return dict(n_atoms=n, box=m * d, pos=(g + 0.25) * d, vel=np.zeros((n, 3)), mass=np.full(n, 20.0),
                charge=np.where(g.sum(1) % 2 == 0, 1.0, -1.0), lj_sigma=np.ones(n), lj_eps=np.zeros(n),
                bond_ij=np.zeros((0, 2), dtype=np.int32), bond_k=z, bond_r0=z,
                angle_ijk=np.zeros((0, 3), dtype=np.int32), angle_k=z, angle_t0=z,
                excl_ptr=np.zeros(n + 1, dtype=np.int32), excl_idx=np.zeros(0, dtype=np.int32))


def test_ewald_sum_gives_the_madelung_constant_of_rock_salt():
    """Direct part (erfc, minimum image to r_long) + reciprocal part + self term of the Ewald sum of a
    rock-salt lattice = -M C q^2 / d per ion pair with the textbook Madelung constant M = 1.7475645946: pins the
    prefactor, the half-space sum, the k-vectors and the alpha convention of the slow force against the direct one."""
    sysd = _rock_salt()
    n = sysd["n_atoms"]
    o = jo.Oracle(sysd, r_short=1.2, r_long=2.0, r_switch=0.2, r_mid=1.6, skin=0.0, flags=0)   # alpha = 3.8 / r_long
    nk = o.ewald_setup(12.0 * 1.9)        # e^{-36}: the reciprocal tail is far below the erfc(3.8) = 8e-8 of the direct one
    assert nk > 1000
    M = {l.split()[0]: float(l.split()[1]) for l in open(os.path.join(GOLD, "madelung_constants.txt")) if l[0] != "#"}
    e = o.potential(1) + o.potential(5)
    assert abs(e / (-(n / 2) * COUL * M["rocksalt"]) - 1.0) < 2e-7
    f = o.forces(5)
    assert np.abs(f).max() < 1e-9 * COUL          # every ion is a centre of symmetry
    # caesium chloride: two interpenetrating simple-cubic lattices, nearest-neighbour distance sqrt(3)/2 of the cube edge
    a, m = 2.0 / math.sqrt(3.0), 4
    g = np.array([(i, j, k) for i in range(m) for j in range(m) for k in range(m)], dtype=np.float64)
    pos = np.vstack([g * a + 0.1, (g + 0.5) * a + 0.1])
    nn = len(pos)
    cs = dict(sysd, n_atoms=nn, box=m * a, pos=pos, vel=np.zeros((nn, 3)), mass=np.full(nn, 20.0),
              charge=np.r_[np.ones(nn // 2), -np.ones(nn // 2)], lj_sigma=np.ones(nn), lj_eps=np.zeros(nn),
              excl_ptr=np.zeros(nn + 1, dtype=np.int32))
    o2 = jo.Oracle(cs, r_short=1.2, r_long=0.5 * m * a, r_switch=0.2, r_mid=1.6, skin=0.0, flags=0)
    assert o2.ewald_setup(12.0 * 3.8 / (0.5 * m * a)) > 1000
    e2 = o2.potential(1) + o2.potential(5)
    assert abs(e2 / (-(nn / 2) * COUL * M["cscl"]) - 1.0) < 2e-7     # nearest-neighbour distance = 1


def test_slow_force_is_the_gradient_of_reciprocal_plus_exclusion_energy(cfg0):
    """Finite differences of U_rec + U_excl (R-21) on the 648-atom water box; sum of the gradient = 0 (translation
    invariance); the exclusion correction alone against its closed form -C q_i q_j erf(alpha r)/r on one molecule."""
    sysd, run = cfg0
    o = jo.Oracle(sysd, **run)
    assert o.ewald_setup(5.0 * 3.8 / 9.0) > 100    # a short k list keeps the test fast; the identity holds for any list
    g = o.forces(5)
    assert np.abs(g.sum(0)).max() < 1e-9 * np.abs(g).max() * len(g)
    x0 = o.pos
    h = 1e-5
    for (i, k) in ((0, 0), (1, 2), (5, 1), (301, 0)):
        xp, xm = x0.copy(), x0.copy()
        xp[i, k] += h; xm[i, k] -= h
        o.set_state(pos=xp, rebuild=False); ep = o.potential(5)
        o.set_state(pos=xm, rebuild=False); em = o.potential(5)
        assert abs((ep - em) / (2 * h) - g[i, k]) < 1e-6 * max(1.0, abs(g[i, k]))
    # one water molecule alone, no reciprocal vectors at all (k_cut below 2 pi / box): only the exclusion correction is left
    one = dict(sysd, n_atoms=3, **{k: sysd[k][:3] for k in ("pos", "vel", "mass", "charge", "lj_sigma", "lj_eps")},
               bond_ij=sysd["bond_ij"][:2], bond_k=sysd["bond_k"][:2], bond_r0=sysd["bond_r0"][:2],
               angle_ijk=sysd["angle_ijk"][:1], angle_k=sysd["angle_k"][:1], angle_t0=sysd["angle_t0"][:1],
               excl_ptr=sysd["excl_ptr"][:4], excl_idx=sysd["excl_idx"][:sysd["excl_ptr"][3]])
    assert np.all(one["excl_idx"] < 3)
    o1 = jo.Oracle(one, **run)
    assert o1.ewald_setup(0.9 * 2 * math.pi / sysd["box"]) == 0
    assert o1.potential(5) == 0.0                                    # no reciprocal vector: the slow force is switched off
    assert o1.ewald_setup(1.01 * 2 * math.pi / sysd["box"]) == 3     # the three shortest half-space vectors
    alpha = 3.8 / run["r_long"]
    q, x = one["charge"], one["pos"]
    excl = sum(-COUL * q[i] * q[j] * special.erf(alpha * np.linalg.norm(x[i] - x[j])) / np.linalg.norm(x[i] - x[j])
               for i, j in ((0, 1), (0, 2), (1, 2)))
    self_e = -COUL * alpha / math.sqrt(math.pi) * (q ** 2).sum()
    V = sysd["box"] ** 3
    rec = 0.0
    for d in range(3):
        k = 2 * math.pi / sysd["box"]
        S = (q * np.exp(1j * k * x[:, d])).sum()
        rec += COUL / V * 4 * math.pi / k ** 2 * math.exp(-k ** 2 / (4 * alpha ** 2)) * abs(S) ** 2
    assert abs(o1.potential(5) - (excl + self_e + rec)) < 1e-10 * abs(excl)


def test_respa1_reductions_and_energy_conservation(relaxed_small):
    """JUMP-RESPA1 (R-21).  (i) Without charges the slow force vanishes and the three-level scheme is
    the two-level one (R-12, paper placement) run n_mid times, bit for bit.  (ii) BAOAB-RESPA1 (comparator) at gamma = 0
    conserves K + U_direct + U_rec + U_excl with an error of second order in the time steps."""
    sysd, run = relaxed_small
    neutral = dict(sysd, charge=np.zeros_like(sysd["charge"]))
    a = jo.Oracle(neutral, **dict(run, flags=2, n_inner=2))
    b = jo.Oracle(neutral, **dict(run, flags=2 | 8, n_inner=2))
    assert a.ewald_setup() > 0
    a.jump_respa1_step(2, 3); b.jump_respa_step(6)
    assert np.array_equal(a.pos, b.pos) and np.array_equal(a.vel, b.vel)
    drift = []
    for dt in (0.25, 0.125):
        o = jo.Oracle(sysd, **dict(run, dt_fs=dt, gamma_per_ps=0.0, flags=16, n_inner=2))
        o.ewald_setup()
        e = []
        for _ in range(int(20 / (4 * dt))):
            o.jump_respa1_step(1, 2)
            e.append(o.kinetic() + o.potential(1) + o.potential(5))
        drift.append(np.std(e))
    assert drift[0] < 0.05 * 192 * KB * 300
    assert 2.5 < drift[0] / drift[1] < 6.5
    # the jumps of the middle level: proposals per unit time do not depend on how the levels are split
    rate = []
    for n_inner, n_mid in ((2, 2), (4, 1)):
        o = jo.Oracle(sysd, **dict(run, flags=1, n_inner=n_inner))
        o.ewald_setup(3.0 * 3.8 / run["r_long"])
        o.jump_respa1_step(40 // (n_inner * n_mid), n_mid)
        rate.append(o.stats()["proposals"] / 40.0)
    assert abs(rate[0] / rate[1] - 1.0) < 0.1


# ---------------------------------------------------------------- NEXT-4: velocity autocorrelation and its spectrum
def test_vacf_of_the_O_step_is_exponential_and_its_spectrum_lorentzian():
    """Free particles under the O part alone are an exact Ornstein-Uhlenbeck process: C(tau) = (3 k_B T / m)
    exp(-gamma tau); the windowed cosine transform of exp(-gamma tau) is the Lorentzian gamma / (gamma^2 + omega^2)."""
    sysd = _ideal_gas(n=6000, seed=3)
    rng = np.random.default_rng(11)
    sysd = dict(sysd, vel=rng.normal(size=(6000, 3)) * np.sqrt(KB * 300 * KCAL / sysd["mass"])[:, None])
    gamma, dt = 5.0, 2.0e-3
    o = jo.Oracle(sysd, r_short=4.0, r_long=6.0, r_mid=5.0, skin=0.5, nlist_every=50, dt_fs=dt * 1e3, gamma_per_ps=gamma,
                  flags=0, seed=9)
    heavy = sysd["mass"] == 16.0
    v0 = o.vel
    c = [jo.velocity_autocorrelation(v0, v0, heavy)]
    for _ in range(60):
        o.baoab_step(5)
        c.append(jo.velocity_autocorrelation(v0, o.vel, heavy))
    c = np.array(c)
    tau = np.arange(61) * 5 * dt
    c0 = 3 * KB * 300 * KCAL / 16.0
    assert abs(c[0] / c0 - 1) < 0.05
    assert np.abs(c / c[0] - np.exp(-gamma * tau)).max() < 0.05          # 3000 atoms: 1/sqrt(9000) = 0.01 per point
    # the transform on an exact exponential
    tt = np.arange(4000) * 1e-3
    om = np.array([0.0, 2.0, 5.0, 12.0])
    spec = jo.vacf_spectrum(np.exp(-gamma * tt), 1e-3, om)
    assert np.abs(spec / (gamma / (gamma ** 2 + om ** 2)) - 1).max() < 0.02
    # one harmonic mode shows up as a line at its frequency
    line = jo.vacf_spectrum(np.cos(7.0 * tt), 1e-3, np.linspace(0.0, 14.0, 57))
    assert abs(np.linspace(0.0, 14.0, 57)[np.argmax(line)] - 7.0) < 0.3


# ------------------------------------------------------------------------------------ NEXT-3: the combined mechanism (R-22)
def test_combined_mechanism_drift_is_the_whole_long_gradient():
    """R-22 (a jump mechanism per force piece F_ij; "both combined"): with F_COMBINED step (C')
    runs ONE mechanism per pair whose F_ij is the sum of the long Coulomb and the long LJ gradient.  The mean-drift
    identity (rate (6) x mean kick (7) = -F_ij/m) must then hold with the SUM: two like charges (Coulomb
    repulsive, -1.9 kcal/mol/A along the pair axis) with a strong LJ attraction (+0.76) -- a dropped term gives -1.9 or
    +0.76 and a sign error +-2.7 instead of -1.1."""
    z = np.zeros(0)
    sysd = dict(n_atoms=2, box=24.0, pos=np.array([[5.0, 5.0, 5.0], [10.0, 5.0, 5.0]]), vel=np.zeros((2, 3)),
                mass=np.array([16.0, 12.0]), charge=np.array([0.5, 0.5]), lj_sigma=np.array([3.4, 3.4]),
                lj_eps=np.array([2.0, 2.0]), bond_ij=np.zeros((0, 2), dtype=np.int32), bond_k=z, bond_r0=z,
                angle_ijk=np.zeros((0, 3), dtype=np.int32), angle_k=z, angle_t0=z,
                excl_ptr=np.zeros(3, dtype=np.int32), excl_idx=np.zeros(0, dtype=np.int32))
    kw = dict(r_short=4.0, r_long=8.0, r_mid=6.0, skin=0.5, ewald_alpha=0.2, eps_jump=0.7, nlist_every=10 ** 9, seed=78)
    parts = {}
    for name, flags in (("coul", 1), ("both", 1 | 2)):          # forces(2): the long gradient the flags hand to the jumps
        o = jo.Oracle(sysd, flags=flags, **kw)
        parts[name] = o.forces(2)
        o.close()
    Fc, F = parts["coul"][:, 0], parts["both"][:, 0]
    assert Fc[0] > 1.0 and (F - Fc)[0] < -0.4 and F[0] > 0.5      # gradient on atom 0: Coulomb +, LJ -, sum +
    o = jo.Oracle(sysd, flags=1 | 2 | jo.F_COMBINED, **kw)
    kT = KB * 300
    sbm = np.sqrt(sysd["mass"] / (kT * KCAL))
    eps = kw["eps_jump"]
    rate0 = max(jo.jump_rate(eps, 1 / kT, sbm[i], abs(F[i]), 0.0) for i in range(2))
    H = 0.02 / (rate0 * math.sqrt(1 + eps * eps))
    rng = np.random.default_rng(9)
    R = 200_000
    acc = np.zeros((2, 3))
    V = rng.normal(size=(R, 2, 3)) / sbm[None, :, None]
    for rep in range(R):
        o.set_vel(V[rep])
        o.jump_half(H, with_accel=False, step=rep)
        acc += o.vel - V[rep]
    mean = acc / R
    pred = -H * KCAL * parts["both"] / sysd["mass"][:, None]
    st = o.stats()
    assert st["accepts"] > 2000 and st["max_g_over_L"] <= 1.0 and st["max_p"] <= 1.0
    for i in range(2):
        assert abs(mean[i, 0] / pred[i, 0] - 1.0) < 0.08, (i, mean[i, 0], pred[i, 0])
        assert np.abs(mean[i, 1:]).max() < 0.06 * abs(pred[i, 0])


def test_combined_mechanism_event_log_and_bounds(relaxed_small):
    """R-22: one chain per atom and half-phase (stream 1 / 4), none in the (J') streams; ring codes 8-10; the bound of a
    ring is the sum of the Coulomb and the LJ bound and dominates the combined gradient of every proposal; more proposals
    than the Coulomb mechanism alone (and more than the two side by side: the LJ bound now also carries the (1/eps)
    term of the general mechanism's rate bound, which BPS does not have)."""
    sysd, kw = _frozen(relaxed_small, flags=1 | 2 | 4 | jo.F_COMBINED, eps_jump=1.0)
    o = jo.Oracle(sysd, **kw)
    o.jump_step(40)
    ev, st = o.events(), o.stats()
    assert st["max_p"] <= 1.0 and st["max_g_over_L"] <= 1.0
    prop = ev[ev["ring"] >= 0]
    assert len(prop) == st["proposals"] > 300 and set(np.unique(prop["ring"])) <= {8, 9, 10}
    assert set(np.unique(ev["stream"])) <= {1, 4}
    assert np.array_equal(prop["accepted"] == 1, prop["U"] <= prop["p"])
    n_comb = st["proposals"]
    counts = {}
    for name, flags in (("coul", 1 | 4), ("two", 1 | 2 | 4)):
        o2 = jo.Oracle(sysd, **dict(kw, flags=flags))
        o2.jump_step(40)
        counts[name] = o2.stats()["proposals"]
    assert counts["coul"] < n_comb < 2 * counts["two"]


def test_mean_square_displacement_of_free_flight_is_v2_t2():
    """NEXT-4: the mean-square displacement on unwrapped positions.  Non-interacting atoms (no charge, no LJ, no bonds)
    without friction fly straight: MSD(t) = <|v|^2> t^2 exactly, also after every atom has left the periodic box several
    times (on wrapped positions it would saturate at the box size); a subset selects."""
    n = 96
    rng = np.random.default_rng(31)
    z = np.zeros(0)
    box = 12.0
    sysd = dict(n_atoms=n, box=box, pos=rng.uniform(0, box, (n, 3)), vel=rng.normal(size=(n, 3)) * 30.0,
                mass=np.full(n, 12.0), charge=np.zeros(n), lj_sigma=np.ones(n), lj_eps=np.zeros(n),
                bond_ij=np.zeros((0, 2), dtype=np.int32), bond_k=z, bond_r0=z, angle_ijk=np.zeros((0, 3), dtype=np.int32),
                angle_k=z, angle_t0=z, excl_ptr=np.zeros(n + 1, dtype=np.int32), excl_idx=np.zeros(0, dtype=np.int32))
    o = jo.Oracle(sysd, r_short=3.0, r_long=5.0, r_mid=4.0, skin=0.5, nlist_every=5, dt_fs=2.0, gamma_per_ps=0.0, flags=3, seed=3)
    x0, v0 = o.pos_unwrapped, o.vel
    o.jump_step(1000)                                   # 2 ps at 30 A/ps: 60 A, five box lengths
    t = 2.0
    sel = np.arange(n) % 3 == 0
    assert np.abs(o.pos).max() <= box and np.abs(o.pos_unwrapped - x0).max() > 3 * box
    assert jo.mean_square_displacement(x0, o.pos_unwrapped) == pytest.approx((v0 ** 2).sum(1).mean() * t * t, rel=1e-9)
    assert jo.mean_square_displacement(x0, o.pos_unwrapped, sel) == pytest.approx((v0[sel] ** 2).sum(1).mean() * t * t, rel=1e-9)
    assert jo.mean_square_displacement(x0, o.pos) < 3 * box * box < jo.mean_square_displacement(x0, o.pos_unwrapped)
