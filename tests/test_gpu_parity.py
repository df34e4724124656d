"""Parity of the CUDA path (through the C ABI) against the fp64 oracle on the same seeded inputs.

Tolerances (BASELINE.json north_star): per-atom force pieces <= 1e-5 relative
(|dF_i| / max(|F_i|, F_rms)), trajectories <= 1e-4 A over 100 steps, integer fields of the event log
bit-exact, T / p / G~ of each event to fp32 rounding.  Trajectory parity is asserted on the window
before the oracle's first fragile decision (R-17).
"""
import numpy as np
import pytest

from paper_2412_15073_b200 import workloads as wl

pytestmark = pytest.mark.gpu

F_TOL = 1e-5
X_TOL = 1e-4


@pytest.fixture(scope="module")
def jb():
    from paper_2412_15073_b200 import binding
    binding.lib()          # fails loudly if the CUDA library is missing
    return binding


@pytest.fixture(scope="module")
def jo():
    from oracle import jump_oracle
    return jump_oracle


@pytest.fixture(scope="module")
def cfg0():
    return wl.make_config(0)


def rel_force_err(fg, fo):
    fg = np.asarray(fg, np.float64)
    frms = np.sqrt((fo ** 2).sum(1).mean())
    return float((np.linalg.norm(fg - fo, axis=1) / np.maximum(np.linalg.norm(fo, axis=1), frms)).max())


def pos_err(g, o, box):
    d = g.pos.cpu().numpy().astype(np.float64) - o.pos
    d -= box * np.round(d / box)
    return float(np.abs(d).max())


def fragile(o):
    """True once the oracle has taken a decision the fp32 path may legitimately take the other way (R-17): an
    accept / expiry / sampler test within 1e-6 of its threshold, or a list-membership / cell decision within 2e-6 A
    of its edge.  After that the two runs are both valid samples of the process but no longer the same one."""
    st = o.stats()
    return st["min_margin"] < 1e-6 or st["min_list_margin"] < 2e-6


INT_FIELDS = ("step", "stream", "atom", "iter", "ring", "j", "accepted", "n_gt")


def check_events(eg, eo, steps=1):
    """R-18: integer fields bit-exact; U exact (R-15).  T = E / lambda-bar carries the relative error of B_v, i.e. of the
    fp32 velocities, and p, G~ are smooth functions of positions (held in fp32 by the pair arithmetic: 1e-5 A at a
    100 A box) and velocities: the two paths drift apart by fp32 rounding, about 1e-7 relative per step (measured:
    1.3e-5 in T after 10 steps at 12 000 atoms, 2e-4 after 100 steps at 648; SURVEY R-18 guessed a flat 1e-5).  Asserted:
    T to 5e-5 relative, p to 1e-4, G~ to 2e-4, each times the number of 10-step chunks elapsed."""
    k = max(1, (steps + 9) // 10)
    assert len(eg) == len(eo)
    for f in INT_FIELDS:
        assert (eg[f] == eo[f]).all(), f
    fin = np.isfinite(eo["T"])
    assert (np.isfinite(eg["T"]) == fin).all()
    if fin.any():   # (a kick that nearly cancels v leaves a small |v| with a large RELATIVE error: the rare outliers)
        rel = np.abs(eg["T"][fin] / eo["T"][fin] - 1)
        assert np.quantile(rel, 0.999) < 5e-5 * k and rel.max() < 5e-3
    if len(eo) == 0:
        return
    assert (eg["U"] == eo["U"].astype(np.float32)).all()       # uniforms are exact in fp32 (R-15)
    # a pair within rounding of a ring edge (force through this ring or not) or a G~ drawn from the other proposal family
    # is a close call that may go the other way without changing any integer of the log (R-17): compared elsewhere
    safe = eo["margin"] >= 2e-6 * steps
    assert safe.mean() > 0.95
    assert np.abs(eg["p"] - eo["p"])[safe].max(initial=0.0) < 1e-4 * k
    assert np.abs(eg["gt"] - eo["gt"])[safe].max(initial=0.0) < 2e-4 * k


def first_divergence(eg, eo):
    """Index of the first logged event (canonical order) whose integer fields differ, None if the logs agree."""
    m = min(len(eg), len(eo))
    bad = np.zeros(m, bool)
    for f in INT_FIELDS:
        bad |= eg[f][:m] != eo[f][:m]
    if bad.any():
        return int(np.argmax(bad))
    return None if len(eg) == len(eo) else m


def divergence_is_a_close_call(eo, k, o, steps):
    """R-17: the two paths may take a discontinuous decision differently only where it is a closer call than they
    differ.  The oracle logs the margin of every decision of every chain iteration (and of the list builds): the
    chain the first differing event belongs to, up to that event, or the lists of the chunk, must show a margin below
    2e-6 times the steps elapsed (the paths drift apart by about 1e-7 per step, relative; 20 times that)."""
    tol = 2e-6 * steps
    e = eo[min(k, len(eo) - 1)]
    chain = eo[(eo["step"] == e["step"]) & (eo["stream"] == e["stream"]) & (eo["atom"] == e["atom"]) & (eo["iter"] <= e["iter"])]
    return (len(chain) and chain["margin"].min() < tol) or o.stats()["min_list_margin"] < tol


# ------------------------------------------------------------------------------------- rows, bounds
def test_bounds_match(jb, jo, cfg0):
    sysd, run = cfg0
    g, o = jb.JumpSim(sysd, **run), jo.Oracle(sysd, **run)
    bg, bo = g.bounds(), o.bounds()
    for k in bo:
        assert bg[k] == pytest.approx(bo[k], rel=1e-12, abs=1e-300), k


@pytest.mark.parametrize("case", ["cfg0", "small5", "no_ring", "big_cells"])
def test_rows_identical(jb, jo, cfg0, case):
    """a1-a3: sort + row build + cell universe (R-10c).  Row A, row B and the universe of ring C must hold the same atoms
    in the same (canonical) order as the oracle's."""
    if case == "cfg0":
        sysd, run = cfg0
    else:
        sysd = wl.small_water(5, seed=11)                      # 375 atoms, box 15.5 A: ragged, several cells
        run = dict(cfg0[1], r_short=4.0, r_long=7.5, r_mid=5.0, seed=5)
        if case == "no_ring":
            run["r_mid"] = 0.0
        if case == "big_cells":
            run["cell_edge"] = 6.1
    g, o = jb.JumpSim(sysd, **run), jo.Oracle(sysd, **run)
    nM, nL, nV = o.row_counts()
    for i in range(g.n):
        for which, cnt in ((1, nM), (2, nL), (3, nV)):
            rg = g.row(which, i)
            assert len(rg) == cnt[i]
            if i % 5 == 0:
                assert (rg == o.row(which - 1, i)).all()
    st = g.stats()
    assert st["error"] == 0 and all(m <= c for m, c in zip(st["max_row"], st["cap_row"]) if c)


# ------------------------------------------------------------------------------------- forces
@pytest.mark.parametrize("flags", [3, 1, 0])
def test_force_pieces_cfg0(jb, jo, cfg0, flags):
    """a4, a5, a10: F0, unsplit, long, bonded, short non-bonded; flags=1 keeps the LJ tail in F0 (R-13)."""
    sysd, run = cfg0
    run = dict(run, flags=flags)
    g, o = jb.JumpSim(sysd, **run), jo.Oracle(sysd, **run)
    for which in range(5):
        fo = o.forces(which)
        err = rel_force_err(g.forces(which).cpu().numpy(), fo)
        assert err <= F_TOL, (which, err)
    ek, ep = g.energy()
    assert ek == pytest.approx(o.kinetic(), rel=1e-6)
    assert ep == pytest.approx(o.potential(1), rel=1e-5, abs=1e-3)


def test_forces_after_dynamics_and_refresh(jb, jo, cfg0):
    """Forces at a liquid-like (not lattice) geometry, fed in through jump_refresh."""
    sysd, run = cfg0
    o = jo.Oracle(sysd, **run)
    o.baoab_step(300)
    s2 = dict(sysd, pos=np.float32(o.pos).astype(np.float64), vel=np.float32(o.vel).astype(np.float64))
    g, o2 = jb.JumpSim(sysd, **run), jo.Oracle(s2, **run)
    import torch
    g.pos.copy_(torch.as_tensor(np.float32(s2["pos"])))
    g.vel.copy_(torch.as_tensor(np.float32(s2["vel"])))
    g.refresh()
    for which in range(5):
        err = rel_force_err(g.forces(which).cpu().numpy(), o2.forces(which))
        assert err <= F_TOL, (which, err)


def test_forces_solute_config3(jb, jo):
    """Heterogeneous charges and LJ parameters, chain exclusions (1-2, 1-3), 23 558 atoms."""
    sysd, run = wl.make_config(3)
    g, o = jb.JumpSim(sysd, **run), jo.Oracle(sysd, **run)
    for which in (0, 2, 3):
        err = rel_force_err(g.forces(which).cpu().numpy(), o.forces(which))
        assert err <= F_TOL, (which, err)
    nM, nL, nV = o.row_counts()
    for i in list(range(0, 2500, 97)) + list(range(2500, g.n, 1999)):
        for which, cnt in ((1, nM), (2, nL), (3, nV)):
            rg = g.row(which, i)
            assert len(rg) == cnt[i] and (rg == o.row(which - 1, i)).all()


# ------------------------------------------------------------------------------------- jump chains
# Philox keys: for each mechanism the three most robust seeds of 3000..3199 by the oracle's own audit of its decisions
# (tests/golden/scan_parity_seeds.py, oracle only).  Over 100 steps a 648-atom box takes ~2e5 discontinuous decisions
# and rebuilds its lists 25 times; the two paths drift apart by fp32 rounding (~1e-5 A after 100 steps), so on about
# half of all seeds one decision is eventually a closer call than that and is (legitimately, R-17) taken differently.
PARITY_SEEDS = {(1.0, 0): (3055, 3003, 3039), (0.3, 0): (3037, 3038, 3060), (float("inf"), 0): (3042, 3048, 3038),
                (2.0, 1): (3115, 3157, 3038)}   # (adaptive: every seed scores ~1e-9, the scan cannot rank them; kept from the 3000..3199 scan)
COMBINED_SEEDS = (3018, 3054, 3057)   # (scan of seeds 3000..3079 under the round-2 list contract)


def run_parity_window(jb, jo, sysd, run, lanes, n_chunks=10):
    """Both paths, 10 steps at a time with every proposal logged.  Returns the number of steps over which the event
    logs were identical and the positions within X_TOL; a divergence must be a close call of the oracle's (R-17)."""
    g, o = jb.JumpSim(sysd, **run), jo.Oracle(sysd, **run)
    g.set_lanes(lanes)
    window, n_ev, n_acc, rings = 0, 0, 0, set()
    for chunk in range(n_chunks):
        o.reset_stats()
        g.jump_step(10); g.sync(); o.jump_step(10)
        eg, eo = g.events(), o.events()
        k = first_divergence(eg, eo)
        if k is not None:
            assert divergence_is_a_close_call(eo, k, o, window + 10), (window, k, eo[max(0, k - 2):k + 2], eg[max(0, k - 2):k + 2])
            break
        check_events(eg, eo, steps=window + 10)
        assert pos_err(g, o, sysd["box"]) <= X_TOL
        window += 10
        n_ev += len(eo); n_acc += int(eo["accepted"].sum()); rings |= set(np.unique(eo["ring"]).tolist())
        g.clear_events(); o.clear_events()
    sg = g.stats()
    assert sg["error"] == 0 and sg["max_p"] <= 1.0 + 1e-4 and sg["max_g_over_L"] <= 1.0 + 1e-4
    if window == 10 * n_chunks:
        assert np.abs(g.vel.cpu().numpy() - o.vel).max() < 5e-3
    g.close(); o.close()
    return window, n_ev, n_acc, rings


@pytest.mark.parametrize("lanes", [0, 1, 4, 8, 16])
@pytest.mark.parametrize("eps,mode", [(1.0, 0), (0.3, 0), (float("inf"), 0), (2.0, 1)])
def test_event_log_and_trajectory_cfg0(jb, jo, cfg0, eps, mode, lanes):
    """a6-a8: every proposal of 100 JUMP steps (C', J', both halves) equals the oracle's -- partner, ring, accept flag,
    sampler attempts bit for bit, times and probabilities to fp32 rounding -- and the trajectory stays within 1e-4 A
    over the 100 steps (BASELINE.json north_star), for every instantiation of the update kernel (lanes per chain 1, 4,
    8, 16; 0 = the automatic choice, 16 at this size).  Every recorded seed is run; each must agree up to a decision
    that the oracle itself marks as a close call, and at least one must go the whole 100 steps.
    mode 1: adaptive eps(x) = eps0 |F_ij(x)| (NEXT-1, R-19)."""
    if lanes not in (0, 1) and (eps, mode) != (1.0, 0):
        pytest.skip("lane counts 4, 8, 16 are compared on one mechanism")
    sysd, run = cfg0
    best = 0
    for seed in PARITY_SEEDS[(eps, mode)]:
        r = dict(run, flags=jb.F_COUL_JUMPS | jb.F_LJ_JUMPS | jb.F_EVENT_LOG, eps_jump=eps, eps_mode=mode, seed=seed)
        window, n_ev, n_acc, rings = run_parity_window(jb, jo, sysd, r, lanes)
        assert window >= 10
        if window == 100:
            assert n_ev > 150000 and rings == {-1, 0, 1, 2, 4, 5, 6}
            assert mode == 0 or n_acc > 30000           # the adaptive mechanism accepts about a quarter of its proposals
        best = max(best, window)
        if best == 100:
            break
    # the adaptive mechanism accepts a quarter of its proposals (four G~ draws and kicks per atom and step): no seed of
    # the range keeps every one of its ~1e5 sampler decisions away from its thresholds for 100 steps
    assert best == 100 or (mode == 1 and best >= 40)


def test_bjaoajb_scheme_matches_oracle(jb, jo, cfg0):
    """NEXT-3: B J A O A J B as the scheme of jump_step -- event log and trajectory against the oracle,
    and without any jump mechanism the scheme is bitwise the C' scheme without jumps (BAOAB with F0)."""
    sysd, run = cfg0
    r = dict(run, flags=jb.F_COUL_JUMPS | jb.F_LJ_JUMPS | jb.F_EVENT_LOG | jb.F_BJAOAJB, seed=3065)   # scan_parity_seeds.py
    g, o = jb.JumpSim(sysd, **r), jo.Oracle(sysd, **r)
    g.jump_step(10); g.sync(); o.jump_step(10)
    assert len(o.events()) > 15000
    check_events(g.events(), o.events())
    g.clear_events(); o.clear_events()
    g.jump_step(10); g.sync(); o.jump_step(10)
    if not fragile(o):
        assert pos_err(g, o, sysd["box"]) <= X_TOL
        assert np.abs(g.vel.cpu().numpy() - o.vel).max() < 5e-3
    a, b = jb.JumpSim(sysd, **dict(run, flags=jb.F_BJAOAJB)), jb.JumpSim(sysd, **dict(run, flags=0))
    a.jump_step(25); b.jump_step(25); a.sync(); b.sync()
    assert (a.pos == b.pos).all() and (a.vel == b.vel).all() and a.stats()["proposals"] == 0


@pytest.mark.parametrize("lanes", [0, 1])
def test_combined_mechanism_matches_oracle(jb, jo, cfg0, lanes):
    """NEXT-3 (R-22): JUMP_F_COMBINED -- one mechanism per pair for the whole long pair gradient (Coulomb + LJ) in step C',
    no step J': every proposal of up to 100 steps equals the oracle's (partner, ring code 8-10, accept flag, sampler
    attempts), trajectory within 1e-4 A, up to a decision the oracle marks as a close call; and the flag is refused
    without both jump flags."""
    sysd, run = cfg0
    flags = jb.F_COUL_JUMPS | jb.F_LJ_JUMPS | jb.F_EVENT_LOG | jb.F_COMBINED
    best = 0
    for seed in COMBINED_SEEDS:
        window, n_ev, n_acc, rings = run_parity_window(jb, jo, sysd, dict(run, flags=flags, seed=seed), lanes)
        assert window >= 10
        if window >= 50:
            assert rings == {-1, 8, 9, 10} and n_ev > 60000 and n_acc > 500
        best = max(best, window)
        if best == 100:
            break
    assert best >= 50
    with pytest.raises(jb.JumpError, match="COMBINED"):
        jb.JumpSim(sysd, **dict(run, flags=jb.F_COUL_JUMPS | jb.F_COMBINED))


def test_jump_half_statistics_frozen_x(jb, jo, cfg0):
    """The C'/J' half-phase alone at frozen x, long duration (many events per atom), with and without drift."""
    sysd, run = cfg0
    run = dict(run, flags=jb.F_COUL_JUMPS | jb.F_LJ_JUMPS | jb.F_EVENT_LOG)
    for accel in (True, False):
        g, o = jb.JumpSim(sysd, **run), jo.Oracle(sysd, **run)
        g.jump_half(0.004, accel, step=7); g.sync(); o.jump_half(0.004, accel, step=7)
        check_events(g.events(), o.events())
        assert np.abs(g.vel.cpu().numpy() - o.vel).max() < 2e-3
        assert (g.pos.cpu().numpy() == np.float32(o.pos)).all()     # x frozen


def test_only_coulomb_jumps_and_only_lj_jumps(jb, jo, cfg0):
    sysd, run = cfg0
    for flags in (1, 2):
        r = dict(run, flags=flags | jb.F_EVENT_LOG)
        g, o = jb.JumpSim(sysd, **r), jo.Oracle(sysd, **r)
        g.jump_step(5); g.sync(); o.jump_step(5)
        check_events(g.events(), o.events())
        assert pos_err(g, o, sysd["box"]) <= X_TOL


# ------------------------------------------------------------------------------------- BAOAB, RESPA
def test_baoab_trajectory_100_steps(jb, jo, cfg0):
    sysd, run = cfg0
    g, o = jb.JumpSim(sysd, **run), jo.Oracle(sysd, **run)
    g.baoab_step(100); g.sync(); o.baoab_step(100)
    assert g.step == 100 == o.step
    assert pos_err(g, o, sysd["box"]) <= X_TOL
    assert np.abs(g.vel.cpu().numpy() - o.vel).max() < 5e-3
    assert rel_force_err(g.forces(0).cpu().numpy(), o.forces(0)) <= 20 * F_TOL    # forces at diverged-by-1e-5-A positions


def test_baoab_energy_conservation_gamma0(jb, cfg0):
    """gamma = 0, jumps off: BAOAB is velocity Verlet; the energy error is O(dt^2) and does not drift."""
    sysd, run = cfg0
    out = []
    for dt in (0.5, 0.25):
        g = jb.JumpSim(sysd, **dict(run, gamma_per_ps=0.0, dt_fs=dt, flags=0))
        g.baoab_step(int(20 / dt))
        e0 = sum(g.energy())
        dev = []
        for _ in range(10):
            g.baoab_step(int(20 / dt))
            dev.append(sum(g.energy()) - e0)
        out.append(np.abs(dev).max())
    assert out[0] < 0.02 * 648 * 0.6          # small against the thermal energy scale
    assert out[1] < 0.5 * out[0]              # second order: quartered, allow 2x


@pytest.mark.parametrize("flags,mode", [(3, 0), (3 | 8, 0), (3 | 16, 0), (3 | 8 | 16, 0), (1, 0), (3, 1), (3 | 8, 1)])
def test_respa_variants(jb, jo, cfg0, flags, mode):
    """a9: JUMP-RESPA (BASELINE variant and the paper's variant) and the BAOAB-RESPA comparator (R-12);
    mode 1: with the adaptive eps of R-19."""
    sysd, run = cfg0
    r = dict(run, flags=flags | jb.F_EVENT_LOG, eps_mode=mode, eps_jump=2.0 if mode else run["eps_jump"])
    g, o = jb.JumpSim(sysd, **r), jo.Oracle(sysd, **r)
    g.jump_respa_step(3); g.sync(); o.jump_respa_step(3)
    assert g.step == 12 == o.step
    eg, eo = g.events(), o.events()
    if flags & 16:
        assert len(eg) == 0 == len(eo)
    elif fragile(o):                       # the rows rebuilt at step 10 may differ by one entry: compare up to there
        keep_g, keep_o = eg["step"] < 2, eo["step"] < 2
        check_events(eg[keep_g], eo[keep_o])
        return
    else:
        check_events(eg, eo)
        assert set(np.unique(eo["stream"])) <= {5, 6, 7, 8} and len(eo) > 1000
    assert pos_err(g, o, sysd["box"]) <= X_TOL
    assert np.abs(g.vel.cpu().numpy() - o.vel).max() < 5e-3


def test_degenerate_no_jumps_is_baoab_with_short_forces(jb, jo, cfg0):
    """flags = 0: jump_step is BAOAB with F0 (C.6 'JUMP degenerate cases'); no events, no proposals."""
    sysd, run = cfg0
    r = dict(run, flags=0)
    g, o = jb.JumpSim(sysd, **r), jo.Oracle(sysd, **r)
    g.jump_step(50); g.sync(); o.jump_step(50)
    assert pos_err(g, o, sysd["box"]) <= X_TOL
    assert g.stats()["proposals"] == 0


def _liquid_state(jo, sysd, run, n_steps=300):
    """A liquid-like (not lattice) state made by the ORACLE (no test input ever comes from the CUDA path), fp32-exact."""
    o = jo.Oracle(sysd, **run)
    o.baoab_step(n_steps)
    s2 = dict(sysd, pos=np.float32(o.pos).astype(np.float64), vel=np.float32(o.vel).astype(np.float64))
    o.close()
    return s2


def test_refresh_lazy_keeps_valid_rows_and_rebuilds_when_needed(jb, jo, cfg0):
    """jump_refresh_lazy: positions moved by less than skin/2 keep the rows (no rebuild, stale cell table) and F0
    equals the oracle's at the new positions; one atom pushed beyond skin/2 triggers the rebuild; either way the next
    steps run without an error flag."""
    import torch
    sysd, run = cfg0
    s2 = _liquid_state(jo, sysd, run)
    g = jb.JumpSim(s2, **run)
    n0 = g.stats()["rebuilds"]
    rng = np.random.default_rng(17)
    pos2 = np.float32(s2["pos"] + rng.uniform(-0.03, 0.03, size=s2["pos"].shape)).astype(np.float64)   # |d| < 0.06: room for 3 more steps below skin/2
    g.pos.copy_(torch.as_tensor(np.float32(pos2)))
    assert g.refresh_lazy() is False and g.stats()["rebuilds"] == n0
    o = jo.Oracle(dict(s2, pos=pos2), **run)
    for which in (0, 2):
        assert rel_force_err(g.forces(which).cpu().numpy(), o.forces(which)) <= F_TOL
    g.jump_step(3); g.sync()
    assert g.stats()["error"] == 0
    pos3 = pos2.copy()
    pos3[5, 0] += 0.8                                       # one atom pushed out of its skin/2 ball
    g.pos.copy_(torch.as_tensor(np.float32(pos3)))
    n1 = g.stats()["rebuilds"]
    g.set_lax_skin(True)                                    # (the pushed atom is shot away by its neighbours)
    assert g.refresh_lazy() is True and g.stats()["rebuilds"] == n1 + 1
    o = jo.Oracle(dict(s2, pos=np.float32(pos3).astype(np.float64)), **run)
    assert rel_force_err(g.forces(0).cpu().numpy(), o.forces(0)) <= F_TOL
    g.jump_step(10); g.sync()
    assert g.stats()["error"] == 0


def test_determinism_bitwise(jb, cfg0):
    """Same inputs and seed: same bits (counter-based RNG, no floating-point atomics, canonical rows)."""
    sysd, run = cfg0
    res = []
    for _ in range(2):
        g = jb.JumpSim(sysd, **run)
        g.jump_step(25); g.jump_respa_step(2); g.sync()
        res.append((g.pos.cpu().numpy().copy(), g.vel.cpu().numpy().copy(), g.stats()["proposals"]))
    assert (res[0][0] == res[1][0]).all() and (res[0][1] == res[1][1]).all() and res[0][2] == res[1][2]


def test_step_batching_is_invisible(jb, cfg0):
    """jump_step(20) == 20 x jump_step(1): the closing/opening half-phases fused across steps are the same maths."""
    sysd, run = cfg0
    a, b = jb.JumpSim(sysd, **run), jb.JumpSim(sysd, **run)
    a.jump_step(20); a.sync()
    for _ in range(20):
        b.jump_step(1)
    b.sync()
    assert (a.pos.cpu().numpy() == b.pos.cpu().numpy()).all() and (a.vel.cpu().numpy() == b.vel.cpu().numpy()).all()


# ------------------------------------------------------------------------------------- edge cases
def test_bad_arguments_are_refused(jb, cfg0):
    sysd, run = cfg0
    for bad in (dict(n_inner=3), dict(r_short=9.5), dict(r_long=9.5), dict(eps_jump=0.0), dict(eps_mode=2),
                dict(eps_mode=1, eps_jump=float("inf")),
                dict(r_switch=0.0), dict(dt_fs=0.0)):
        with pytest.raises(jb.JumpError):
            jb.JumpSim(sysd, **dict(run, **bad))


def test_single_molecule_and_empty_shells(jb, jo):
    """One water in a big box: every row is empty, no proposal is ever made, the step still runs."""
    sysd = wl.water_box(1, 20.0, 3, 4)
    run = dict(wl.make_config(0)[1], flags=3 | 4)
    g, o = jb.JumpSim(sysd, **run), jo.Oracle(sysd, **run)
    g.jump_step(30); g.jump_respa_step(2); g.sync()
    o.jump_step(30); o.jump_respa_step(2)
    assert g.stats()["proposals"] == 0 and pos_err(g, o, sysd["box"]) <= X_TOL
    check_events(g.events(), o.events())


def test_row_overflow_is_reported(jb):
    """A dense cluster in a mostly empty box exceeds the mean-density row capacity: error -3, not silence."""
    sysd = wl.small_water(4, seed=3)
    big = dict(sysd, box=60.0)
    run = dict(wl.make_config(0)[1], r_short=5.0, r_long=9.0)
    with pytest.raises(jb.JumpError, match="-3"):
        jb.JumpSim(big, **run)


# ------------------------------------------------------------------------------------- bench configuration
def check_sampled_rows(g, o, n_sample):
    """Rows M, L, V of a seeded sample of atoms: same atoms, same (canonical) order as the oracle's (bit-exact)."""
    nM, nL, nV = o.row_counts()
    rng = np.random.default_rng(7)
    for i in rng.choice(g.n, size=n_sample, replace=False):
        for which, cnt in ((1, nM), (2, nL), (3, nV)):
            rg = g.row(which, int(i))
            assert len(rg) == cnt[i]
            assert (rg == o.row(which - 1, int(i))).all()


def test_full_size_config1_forces_events_trajectory(jb, jo):
    """BASELINE configs[1] (12 000 atoms), the workload bench.py times: all F0, one logged step, 20 steps."""
    sysd, run = wl.make_config(1)
    run = dict(run, flags=3 | 4)
    g, o = jb.JumpSim(sysd, **run), jo.Oracle(sysd, **run)
    assert rel_force_err(g.forces(0).cpu().numpy(), o.forces(0)) <= F_TOL
    assert rel_force_err(g.forces(1).cpu().numpy(), o.forces(1)) <= F_TOL
    check_sampled_rows(g, o, 48)
    g.jump_step(1); g.sync(); o.jump_step(1)
    check_events(g.events(), o.events())
    g.clear_events(); o.clear_events()
    for n in (9, 10):
        g.jump_step(n); g.sync(); o.jump_step(n)
        g.clear_events(); o.clear_events()
    if not fragile(o):
        assert pos_err(g, o, sysd["box"]) <= X_TOL
    st = g.stats()
    assert st["error"] == 0 and st["max_p"] <= 1 + 1e-4


def test_config2_sampled_forces_and_properties(jb, jo):
    """BASELINE configs[2] (96 000 atoms): F0 against the oracle, Newton's third law of the short part,
    and statistics that hold at any size (p <= 1, |F_ij| <= L, proposals per atom in the expected range)."""
    sysd, run = wl.make_config(2)
    g, o = jb.JumpSim(sysd, **run), jo.Oracle(sysd, **run)
    fo = o.forces(0)
    fg = g.forces(0).cpu().numpy()
    assert rel_force_err(fg, fo) <= F_TOL
    assert np.abs(g.forces(4).cpu().numpy().astype(np.float64).sum(0)).max() < 0.05   # sum of pair gradients = 0
    check_sampled_rows(g, o, 48)   # large grid: multi-block cell scan, two home cells per CTA, cell-centred staging
    g.jump_respa_step(5); g.sync()
    st = g.stats()
    assert st["error"] == 0 and st["max_p"] <= 1 + 1e-4 and st["max_g_over_L"] <= 1 + 1e-4
    per_atom_fs = st["proposals"] / (g.n * 20.0)
    assert 0.5 < per_atom_fs < 20.0


def test_config4_one_million_atoms_properties(jb):
    """BASELINE configs[4] (999 999 atoms, the largest size): no oracle run fits here, so properties that hold at
    any size -- every row within capacity, the pair gradients of the short part sum to zero, thinning bounds hold
    (p <= 1, |F_ij| <= L), proposals per atom in the range of the small boxes, bitwise determinism -- after JUMP
    and JUMP-RESPA steps across a list rebuild (multi-block cell scan, two home cells per build CTA)."""
    sysd, run = wl.make_config(4)
    out = []
    for rep in range(2):
        g = jb.JumpSim(sysd, **run)
        if rep == 0:
            f = g.forces(4).cpu().numpy().astype(np.float64)
            frms = np.sqrt((f ** 2).sum(1).mean())
            assert np.abs(f.sum(0)).max() < 1e-4 * frms * np.sqrt(g.n)      # Newton's third law up to fp32 rounding
        g.jump_step(12); g.jump_respa_step(2); g.sync()
        st = g.stats()
        assert st["error"] == 0 and st["rebuilds"] >= 2
        assert st["max_p"] <= 1 + 1e-4 and st["max_g_over_L"] <= 1 + 1e-4
        assert all(m <= c for m, c in zip(st["max_row"], st["cap_row"]) if c)
        assert 2.0 < st["proposals"] / (g.n * 20.0) < 20.0
        out.append((g.pos.cpu().numpy().copy(), g.vel.cpu().numpy().copy()))
        g.close()
    assert (out[0][0] == out[1][0]).all() and (out[0][1] == out[1][1]).all()


def test_config4_forces_rows_and_one_outer_step_against_the_oracle(jb, jo):
    """BASELINE configs[4], the workload and launch configuration bench.py times (999 999 atoms, JUMP-RESPA 1:4 fs, one
    lane per chain, multi-kernel sort, resident-grid list kernels): F0 of EVERY atom against the oracle's, rows A and B
    and the cell universe of a seeded sample of atoms bit for bit, then one JUMP-RESPA outer step (four inner steps,
    ~2.5e7 discontinuous decisions): the same number of proposals and accepted jumps up to the handful of close calls
    the fp32 path may take the other way (R-17), and the positions of all but those atoms within 1e-4 A."""
    sysd, run = wl.make_config(4)
    g, o = jb.JumpSim(sysd, **run), jo.Oracle(sysd, **run)
    assert rel_force_err(g.forces(0).cpu().numpy(), o.forces(0)) <= F_TOL
    check_sampled_rows(g, o, 64)
    g.jump_respa_step(1); g.sync(); o.jump_respa_step(1)
    sg, so = g.stats(), o.stats()
    assert sg["error"] == 0 and sg["max_p"] <= 1 + 1e-4 and sg["max_g_over_L"] <= 1 + 1e-4
    assert so["proposals"] > 4e6 and abs(sg["proposals"] - so["proposals"]) <= 50
    assert so["accepts"] > 1e5 and abs(sg["accepts"] - so["accepts"]) <= 50
    d = g.pos.cpu().numpy().astype(np.float64) - o.pos
    d -= sysd["box"] * np.round(d / sysd["box"])
    bad = np.abs(d).max(1) > X_TOL
    assert bad.sum() <= 50, int(bad.sum())                    # (a jump taken on one side only moves its atom by ~1e-2 A)
    g.close(); o.close()


def test_config2_logged_step_single_lane_chains(jb, jo):
    """BASELINE configs[2] (96 000 atoms), where the update kernel runs one lane per chain -- the instantiation the
    large-box throughput is quoted on: every proposal of one logged JUMP step against the oracle's."""
    sysd, run = wl.make_config(2)
    run = dict(run, flags=3 | 4)
    g, o = jb.JumpSim(sysd, **run), jo.Oracle(sysd, **run)
    g.jump_step(1); g.sync(); o.jump_step(1)
    eo = o.events()
    assert len(eo) > 500000 and set(np.unique(eo["ring"])) == {-1, 0, 1, 2, 4, 5, 6}
    check_events(g.events(), eo)
    assert pos_err(g, o, sysd["box"]) <= X_TOL
    sg, so = g.stats(), o.stats()
    assert sg["error"] == 0 and sg["proposals"] == so["proposals"] and sg["accepts"] == so["accepts"]


def test_config3_solute_logged_steps(jb, jo):
    """BASELINE configs[3] (chain beads with up to five bonded terms each, per-bead charges and LJ parameters): the
    per-atom bonded kernel of the step path, the LJ bounds over a range of sigma, four lanes per chain.  The generator
    leaves the chain on lattice sites with stretched bonds and overlapping beads (a far-from-equilibrium start: forces of
    1e4 kcal/mol/A), so the steps are short (0.25 fs), the lists are rebuilt at every step and the skin check is off;
    parity does not need an equilibrated system: bonded and F0 gradients, then every proposal of 4 logged JUMP steps."""
    sysd, run = wl.make_config(3)
    run = dict(run, flags=3 | 4 | jb.F_LAX_SKIN, nlist_every=1, dt_fs=0.25)
    g, o = jb.JumpSim(sysd, **run), jo.Oracle(sysd, **run)
    for which in (3, 0):
        err = rel_force_err(g.forces(which).cpu().numpy(), o.forces(which))
        assert err <= F_TOL, (which, err)
    done = 0
    for _ in range(4):
        g.jump_step(1); g.sync(); o.jump_step(1)
        eg, eo = g.events(), o.events()
        k = first_divergence(eg, eo)
        if k is not None:                                           # ~1e6 decisions a step on this hot start
            assert divergence_is_a_close_call(eo, k, o, 1)
            break
        check_events(eg, eo)
        assert (eo["ring"] >= 4).sum() > 300                        # LJ chains of the beads and the oxygens
        assert (eo["atom"] < 2500).sum() > 2500                     # chain beads
        assert pos_err(g, o, sysd["box"]) <= X_TOL
        g.clear_events(); o.clear_events()
        done += 1
    assert done >= 1
    sg = g.stats()
    assert sg["error"] == 0 and sg["max_p"] <= 1 + 1e-4 and sg["max_g_over_L"] <= 1 + 1e-4


def test_lists_between_two_builds_against_brute_force(jb, jo, cfg0):
    """Validity of the lists two steps after a build (a conditional build can come from the third step on), against a brute-force O(N^2) search on
    the CURRENT positions rather than against the oracle's own lists: the short list holds every pair closer than r_c,
    rows A and B every pair of their ring, the cell universe every pair closer than r_long; the short-range gradient
    equals the oracle's brute-force sum; a row asked for the first time between two builds (the full list, through
    jump_get_forces(2) and jump_get_energy) gives the brute-force long gradient and energy."""
    sysd, run = cfg0
    s2 = _liquid_state(jo, sysd, run)
    g, o = jb.JumpSim(s2, **run), jo.Oracle(s2, **run)
    assert run["nlist_every"] >= 12
    g.jump_step(2); g.sync(); o.jump_step(2)
    assert g.stats()["rebuilds"] == 1 and not fragile(o)
    x = o.pos; L = sysd["box"]; n = g.n
    d = x[:, None, :] - x[None, :, :]
    d -= L * np.round(d / L)
    r = np.sqrt((d ** 2).sum(-1))
    b = g.bounds()
    rlo, rA, rM, rc, rE = run["r_short"] - run["r_switch"], b["rA"], b["rM"], run["r_short"], run["r_long"]
    eps_r = 1e-5                                            # the two trajectories differ by ~1e-7 A
    for i in range(0, n, 9):
        excl = set(s2["excl_idx"][s2["excl_ptr"][i]:s2["excl_ptr"][i + 1]].tolist()) | {i}
        rows = {w: set(g.row(w, i).tolist()) for w in (0, 1, 2, 3)}
        for w, lo_, hi_ in ((0, 0.0, rc), (1, rlo, rA), (2, rA, rM), (3, 0.0, rE)):
            need = {j for j in range(n) if (w == 3 or j not in excl) and lo_ + eps_r <= r[i, j] < hi_ - eps_r}
            assert need <= rows[w], (i, w, sorted(need - rows[w]))
    assert rel_force_err(g.forces(4).cpu().numpy(), o.forces(4, brute=True)) <= 2 * F_TOL
    assert rel_force_err(g.forces(2).cpu().numpy(), o.forces(2, brute=True)) <= 2 * F_TOL      # full list built just now
    assert g.energy()[1] == pytest.approx(o.potential(1), rel=2e-5, abs=1e-3)
    g.jump_step(5); g.sync()
    assert g.stats()["error"] == 0


def test_displacement_beyond_half_skin_is_an_error_unless_lax(jb, cfg0):
    """List validity is checked on the device at every step (JUMP_E_SKIN): a skin that the fastest atom uses up within
    three steps of a list build (or any time, when there are no rebuilds) is refused at the next synchronising call;
    JUMP_F_LAX_SKIN / jump_set_lax_skin only report it."""
    sysd, run = cfg0
    for kw in (dict(skin=0.12), dict(nlist_every=0)):           # hydrogens: 0.08 A in two steps; no rebuilds at all
        g = jb.JumpSim(sysd, **dict(run, **kw))
        g.jump_step(30)
        with pytest.raises(jb.JumpError, match="-5"):
            g.sync()
    g = jb.JumpSim(sysd, **dict(run, nlist_every=0, flags=run["flags"] | jb.F_LAX_SKIN))
    g.jump_step(30); g.sync()
    assert g.stats()["max_disp"] > 0.5 * run["skin"] and g.stats()["error"] == 0
    g.set_lax_skin(False)
    with pytest.raises(jb.JumpError, match="-5"):
        g.sync()


# ------------------------------------------------------------------------------------- NEXT-4: observables on the device
def test_image_counters_give_continuous_unwrapped_positions(jb, jo, cfg0):
    """Unwrapped positions pos + images * box: equal to the oracle's unwrapped trajectory on the parity window, and
    continuous over a run long enough for many atoms to cross the box faces."""
    sysd, run = cfg0
    box = float(sysd["box"])
    g, o = jb.JumpSim(sysd, **dict(run, seed=3026)), jo.Oracle(sysd, **dict(run, seed=3026))
    g.jump_step(60); g.sync(); o.jump_step(60)
    if not fragile(o):
        assert np.abs(g.pos_unwrapped().cpu().numpy() - o.pos_unwrapped).max() <= X_TOL
    prev = g.pos_unwrapped().cpu().numpy()
    for _ in range(150):                                   # 3 ps, a check every 20 fs
        g.jump_step(20)
        cur = g.pos_unwrapped().cpu().numpy()
        assert np.abs(cur - prev).max() < 2.0              # a missed or doubled image would be a jump of one box length
        prev = cur
    img = g.images().cpu().numpy()
    assert (img != 0).any(1).sum() > 20                    # atoms did cross
    w = g.pos.cpu().numpy().astype(np.float64)
    assert (w >= 0).all() and (w < box).all()
    assert g.refresh_lazy() in (False, True)               # the hand-back call keeps the trajectory: counters survive
    assert (g.images().cpu().numpy() == img).all()
    assert np.abs(g.pos_unwrapped().cpu().numpy() - prev).max() < 1e-5
    g.refresh()
    assert (g.images().cpu().numpy() == 0).all()           # jump_refresh restarts the counters


@pytest.mark.parametrize("cfg,lj_only", [(0, True), (0, False), (1, True)])
def test_rdf_histogram_matches_plain_definition(jb, jo, cfg, lj_only):
    """jump_rdf_accumulate against the oracle's O(N^2) pair histogram of the same positions (integer counts; a pair
    within fp32 rounding of a bin edge may fall on the other side of it).  The positions are a seeded perturbation of
    the generator's, handed over by jump_refresh_lazy WITHOUT a rebuild: the cell table the kernel walks is stale by up
    to skin/2 per atom, as it is between two rebuilds of a run."""
    import torch
    sysd, run = wl.make_config(cfg)
    g = jb.JumpSim(sysd, **run)
    rng = np.random.default_rng(23)
    pos2 = np.float32(sysd["pos"] + rng.uniform(-0.09, 0.09, size=sysd["pos"].shape))   # (oxygens may move 0.167 A)
    g.pos.copy_(torch.as_tensor(pos2))
    assert g.refresh_lazy() is False
    box = float(sysd["box"])
    x = np.mod(pos2.astype(np.float64), box)
    r_max, n_bins = 8.0, 160
    hist = torch.zeros(n_bins, dtype=torch.int64, device=g.device)
    g.rdf_accumulate(hist, r_max, lj_only=lj_only); g.sync()
    sel = np.asarray(sysd["lj_eps"]) > 0 if lj_only else np.ones(g.n, bool)
    ref = jo.pair_histogram(x[sel], box, r_max, n_bins)
    got = hist.cpu().numpy()
    assert abs(int(got.sum()) - int(ref.sum())) <= 2 and np.abs(got - ref).sum() <= 8
    g.rdf_accumulate(hist, r_max, lj_only=lj_only); g.sync()
    assert (hist.cpu().numpy() == 2 * got).all()           # accumulates
    with pytest.raises(jb.JumpError):
        g.rdf_accumulate(hist, 0.51 * box, lj_only=lj_only)


# ------------------------------------------------------------------------------------- orthorhombic boxes
@pytest.mark.parametrize("case", ["small", "config1"])
def test_orthorhombic_box(jb, jo, case):
    """box[3] with three different edges (the ABI's general case; every BASELINE config is cubic): rows, forces,
    event log and a short trajectory against the oracle.  "small": exact-minimum-image build path; "config1": the
    12 000-atom box stretched in y and z (vacuum slabs), cell-centred build path, different cell counts per edge."""
    if case == "small":
        sysd = wl.small_water(5, seed=13)
        box = np.array([16.0, 18.5, 21.0])
        run = dict(wl.make_config(0)[1], r_short=4.0, r_long=7.5, r_mid=5.5, seed=9)
    else:
        sysd, run = wl.make_config(1)
        box = np.array([float(sysd["box"]), 55.0, 61.5])
    sysd = dict(sysd, box=box)
    run = dict(run, flags=3 | 4)
    g, o = jb.JumpSim(sysd, **run), jo.Oracle(sysd, **run)
    check_sampled_rows(g, o, 40)
    for which in (0, 1, 2):
        assert rel_force_err(g.forces(which).cpu().numpy(), o.forces(which)) <= F_TOL, which
    g.jump_step(10); g.sync(); o.jump_step(10)
    eg, eo = g.events(), o.events()
    k = first_divergence(eg, eo)
    if k is not None:
        assert divergence_is_a_close_call(eo, k, o, 10)
    else:
        check_events(eg, eo)
    if k is None and not fragile(o):
        d = g.pos.cpu().numpy().astype(np.float64) - o.pos
        d -= box * np.round(d / box)
        assert np.abs(d).max() <= X_TOL
    assert g.stats()["error"] == 0


# ------------------------------------------------------------------------------------- NEXT-2: slow force, JUMP-RESPA1
@pytest.mark.parametrize("cfg", [0, 3])
def test_slow_force_reciprocal_ewald(jb, jo, cfg):
    """R-21: grad(U_rec + U_excl) and the energy U_rec + U_self + U_excl against the oracle's plain double sum: 648-atom
    water box with the default k_cut = 8 alpha (2 000 vectors, several tiles and a ragged tail in both passes), and the
    23 558-atom solute box (heterogeneous charges, chain exclusions, 16 atom chunks) with a shorter list."""
    sysd, run = wl.make_config(cfg)
    g, o = jb.JumpSim(sysd, **run), jo.Oracle(sysd, **run)
    k_cut = 0.0 if cfg == 0 else 4.0 * 3.8 / run["r_long"]
    nk = g.ewald_setup(k_cut)
    assert nk == o.ewald_setup(k_cut) and nk > 1000
    fo = o.forces(5)
    err = rel_force_err(g.forces(5).cpu().numpy(), fo)
    assert err <= F_TOL, err
    assert g.slow_energy() == pytest.approx(o.potential(5), rel=2e-6)
    if cfg == 0:   # after dynamics (sorted order changed, residuals xl non-zero)
        g.jump_step(25); g.sync(); o.jump_step(25)
        if not fragile(o):
            assert rel_force_err(g.forces(5).cpu().numpy(), o.forces(5)) <= F_TOL


@pytest.mark.parametrize("flags,n_inner,n_mid,mode", [(3, 2, 3, 0), (3 | 16, 2, 3, 0), (1, 2, 2, 0), (3, 2, 3, 1), (3, 4, 1, 0)])
def test_respa1_three_levels(jb, jo, cfg0, flags, n_inner, n_mid, mode):
    """JUMP-RESPA1 (1 : 2 : 6 fs as in the paper's Table 2) and the BAOAB-RESPA1 comparator: event log
    of the middle-level jumps and the trajectory against the oracle; mode 1: with the adaptive eps of R-19 (the paper's
    setting for these runs); n_mid = 1: the slow kick around every middle step."""
    sysd, run = cfg0
    r = dict(run, flags=flags | jb.F_EVENT_LOG, n_inner=n_inner, eps_mode=mode, eps_jump=2.0 if mode else run["eps_jump"])
    g, o = jb.JumpSim(sysd, **r), jo.Oracle(sysd, **r)
    assert g.ewald_setup() == o.ewald_setup()
    n_out = 3
    g.jump_respa1_step(n_out, n_mid); g.sync(); o.jump_respa1_step(n_out, n_mid)
    assert g.step == n_out * n_mid * n_inner == o.step
    eg, eo = g.events(), o.events()
    if flags & 16:
        assert len(eg) == 0 == len(eo)
    elif fragile(o):
        keep_g, keep_o = eg["step"] < 2, eo["step"] < 2
        check_events(eg[keep_g], eo[keep_o])
        return
    else:
        check_events(eg, eo)
        assert len(eo) > 1000
    assert pos_err(g, o, sysd["box"]) <= X_TOL
    assert np.abs(g.vel.cpu().numpy() - o.vel).max() < 5e-3


def test_respa1_needs_setup_and_conserves_energy(jb, cfg0):
    """jump_respa1_step before jump_ewald_setup is refused; BAOAB-RESPA1 at gamma = 0 conserves K + U_direct + U_rec +
    U_excl to second order in the time steps (a wrong sign or factor of the slow kick would show as a drift)."""
    sysd, run = cfg0
    g = jb.JumpSim(sysd, **dict(run, flags=16, n_inner=2))
    with pytest.raises(RuntimeError):
        g.jump_respa1_step(1, 2)
    out = []
    for dt in (0.5, 0.25):
        g = jb.JumpSim(sysd, **dict(run, flags=16, n_inner=2, dt_fs=dt, gamma_per_ps=0.0))
        g.ewald_setup()
        e = []
        for _ in range(int(30 / (4 * dt))):
            g.jump_respa1_step(1, 2)
            ek, ep = g.energy()
            e.append(ek + ep + g.slow_energy())
        out.append(np.std(e))
    assert out[0] < 0.02 * 648 * 0.6
    assert out[1] < 0.5 * out[0]


def test_velocity_autocorrelation_on_the_device(jb, jo, cfg0):
    """NEXT-4: jump_vacf_mark / jump_vacf_dot against the plain definition (oracle.velocity_autocorrelation) on the
    oracle's own velocities of the same seeded run: exact at lag 0 (the generator's fp32 velocities), then along 40 JUMP
    steps -- across a re-sort, which permutes the atoms -- to the accuracy the trajectories agree to (R-16)."""
    sysd, run = cfg0
    g, o = jb.JumpSim(sysd, **run), jo.Oracle(sysd, **run)
    with pytest.raises(RuntimeError):
        g.vacf_dot()
    g.vacf_mark()
    v0 = o.vel
    oxy = sysd["lj_eps"] > 0
    assert g.vacf_dot() == pytest.approx(jo.velocity_autocorrelation(v0, v0), rel=1e-12)
    assert g.vacf_dot(lj_only=True) == pytest.approx(jo.velocity_autocorrelation(v0, v0, oxy), rel=1e-12)
    c0 = jo.velocity_autocorrelation(v0, v0)
    for _ in range(4):
        g.jump_step(10); g.sync(); o.jump_step(10)
        if fragile(o):
            break
        assert abs(g.vacf_dot() - jo.velocity_autocorrelation(v0, o.vel)) < 2e-4 * c0
        assert abs(g.vacf_dot(lj_only=True) - jo.velocity_autocorrelation(v0, o.vel, oxy)) < 2e-4 * c0
    assert o.step >= 10


def test_mean_square_displacement_on_the_device(jb, jo, cfg0):
    """NEXT-4: jump_msd_mark / jump_msd against the plain definition (oracle.mean_square_displacement) on the oracle's own
    unwrapped positions of the same seeded run, along 40 JUMP steps (across re-sorts) to the accuracy the trajectories
    agree to; then over 3 ps, long enough for atoms to cross the box faces, against the same sum formed on the host from
    d_pos and the image counters; the LJ-carrier subset selects the oxygens."""
    sysd, run = cfg0
    g, o = jb.JumpSim(sysd, **run), jo.Oracle(sysd, **run)
    with pytest.raises(RuntimeError):
        g.msd()
    g.msd_mark()
    x0, x0g = o.pos_unwrapped, g.pos_unwrapped().cpu().numpy()
    oxy = sysd["lj_eps"] > 0
    assert g.msd() == 0.0
    for _ in range(4):
        g.jump_step(10); g.sync(); o.jump_step(10)
        if fragile(o):
            break
        want, want_o = jo.mean_square_displacement(x0, o.pos_unwrapped), jo.mean_square_displacement(x0, o.pos_unwrapped, oxy)
        assert g.msd() == pytest.approx(want, rel=2e-3, abs=1e-7) and g.msd(lj_only=True) == pytest.approx(want_o, rel=2e-3, abs=1e-7)
    assert o.step >= 10
    g.jump_step(3000); g.sync()
    xg = g.pos_unwrapped().cpu().numpy()
    assert np.abs(g.images().cpu().numpy()).max() >= 1                      # somebody has left the box
    assert g.msd() == pytest.approx(jo.mean_square_displacement(x0g, xg), rel=1e-5)
    assert g.msd(lj_only=True) == pytest.approx(jo.mean_square_displacement(x0g, xg, oxy), rel=1e-5)
    assert 0.5 < g.msd() < 50.0                                             # A^2 after 3 ps of liquid water


@pytest.mark.parametrize("form", ["blocked", "tables", "direct"])
def test_slow_force_orthorhombic_box_and_both_kernel_forms(jb, jo, form, monkeypatch):
    """R-21 on a box with three different edges (different n_max per dimension: the table offsets and the tile grid of
    the factorised passes) and through every form of the two passes: register-blocked over 4 x 4 tiles (the default),
    one term per thread on the phase-factor tables (JUMP_B200_EWALD_BLOCKED=0), direct sines and cosines
    (JUMP_B200_EWALD_DIRECT=1); a k list of 3 vectors (shorter than a tile) and an empty one."""
    if form == "direct":
        monkeypatch.setenv("JUMP_B200_EWALD_DIRECT", "1")
    if form == "tables":
        monkeypatch.setenv("JUMP_B200_EWALD_BLOCKED", "0")
    sysd = wl.small_water(5, seed=13)
    box = np.array([16.0, 18.5, 21.0])
    run = dict(wl.make_config(0)[1], r_short=4.0, r_long=7.5, r_mid=5.5, seed=9)
    sysd = dict(sysd, box=box)
    g, o = jb.JumpSim(sysd, **run), jo.Oracle(sysd, **run)
    for k_cut in (0.0, 1.05 * 2 * np.pi / 16.0, 0.1):
        nk = g.ewald_setup(k_cut)
        assert nk == o.ewald_setup(k_cut)
        fo = o.forces(5)
        fg = g.forces(5).cpu().numpy().astype(np.float64)
        if nk == 0:
            assert np.abs(fg).max() == 0.0 and np.abs(fo).max() == 0.0 and g.slow_energy() == 0.0
        else:
            assert rel_force_err(fg, fo) <= F_TOL, (k_cut, rel_force_err(fg, fo))
            assert g.slow_energy() == pytest.approx(o.potential(5), rel=2e-6)
