"""Long-run averages of the CUDA JUMP path against CUDA BAOAB and against the fp64 oracle (BASELINE.json
north_star: T, potential energy, RDF and diffusion constant within stated statistical error bars).

JUMP is a different stochastic process from BAOAB with the same invariant measure mu, so realised
trajectories differ and what must agree are averages under mu.  Error bars: standard errors from block averages
(tests/observables.py); a comparison passes when the means differ by less than 4 combined standard errors plus a
stated slack for the O(delta^2) time-step bias, which differs between the two splittings.
"""
import numpy as np
import pytest

from paper_2412_15073_b200 import workloads as wl
import observables as ob

pytestmark = pytest.mark.gpu
KB = 1.987204259e-3


@pytest.fixture(scope="module")
def jb():
    from paper_2412_15073_b200 import binding
    return binding


@pytest.fixture(scope="module")
def jo():
    from oracle import jump_oracle
    jump_oracle.build()
    return jump_oracle


def sample_run(sim, step_fn, energy_fn, pos_fn, n_samples, stride, oxy, snap_every):
    T, U, snaps = [], [], []
    n = len(oxy) * 3
    for k in range(n_samples):
        step_fn(stride)
        ek, ep = energy_fn()
        T.append(2.0 * ek / (3.0 * n * KB))
        U.append(ep / len(oxy))
        if k % snap_every == 0:
            snaps.append(pos_fn()[oxy].astype(np.float64))
    return np.array(T), np.array(U), snaps


def test_long_run_averages_jump_vs_baoab_vs_oracle(jb, jo):
    sysd, run = wl.make_config(0)                       # 216 waters, 648 atoms, box 18.64 A
    box = float(sysd["box"])
    oxy = np.nonzero(np.asarray(sysd["lj_eps"]) > 0)[0]
    assert len(oxy) * 3 == sysd["n_atoms"]
    # every run starts from the generator's lattice state and discards its own burn-in (no test input comes from
    # the CUDA path): 6 ps on the GPU, 2.5 ps of JUMP (whose jumps thermalise within a fraction of a ps) in the oracle
    stride, n_samples, snap_every = 20, 2000, 5          # 40 ps per GPU run, a snapshot every 100 fs
    res = {}
    for name in ("jump", "baoab"):
        g = jb.JumpSim(sysd, **dict(run, seed=run["seed"] + (1 if name == "jump" else 2)))
        step = g.jump_step if name == "jump" else g.baoab_step
        g.baoab_step(3000); step(3000)
        res[name] = sample_run(g, step, g.energy, lambda: g.pos.cpu().numpy(), n_samples, stride, oxy, snap_every)
        st = g.stats()
        assert st["error"] == 0 and st["max_p"] <= 1 + 1e-4
        g.close()
    o = jo.Oracle(sysd, **dict(run, seed=run["seed"] + 3))
    o.jump_step(2500)
    res["oracle"] = sample_run(o, o.jump_step, lambda: (o.kinetic(), o.potential(1)), lambda: o.pos, 200, stride, oxy, 1)
    o.close()

    T = {k: ob.block_mean_se(v[0]) for k, v in res.items()}      # kinetic temperature, K
    U = {k: ob.block_mean_se(v[1]) for k, v in res.items()}      # potential energy, kcal/mol per molecule
    print("T", T, "U", U)
    r, gj, ej = ob.rdf_blocks(res["jump"][2], box, 8.0, 64)      # O-O radial distribution function
    _, gb, eb = ob.rdf_blocks(res["baoab"][2], box, 8.0, 64)
    _, go, eo = ob.rdf_blocks(res["oracle"][2], box, 8.0, 64)
    ps = run["dt_fs"] * 1e-3
    Dj = ob.diffusion_atoms(res["jump"][2], box, stride * snap_every * ps, 2, 10)     # MSD slope between 0.2 and 1 ps
    Db = ob.diffusion_atoms(res["baoab"][2], box, stride * snap_every * ps, 2, 10)
    Do = ob.diffusion_atoms(res["oracle"][2], box, stride * ps, 10, 50)
    print("D", Dj, Db, Do)

    # (1) the CUDA path against the oracle: the SAME process, so every long-run average agrees, the dynamical one too
    assert ob.agree(T["jump"], T["oracle"], 4.0, slack=1.0), (T["jump"], T["oracle"])
    assert ob.agree(U["jump"], U["oracle"], 4.0, slack=0.05), (U["jump"], U["oracle"])
    assert (np.abs(gj - go) <= 4.0 * np.hypot(ej, eo) + 0.15).all(), np.abs(gj - go).max()
    assert ob.agree(Dj, Do, 4.0, slack=0.1 * Dj[0]), (Dj, Do)

    # (2) JUMP against BAOAB: different processes, the same invariant measure mu -- configurational
    # averages agree.  The kinetic temperature read at the end of a step carries each splitting's own O(delta^2) bias
    # (stiff O-H bonds at delta = 1 fs; the jumps resample velocity components exactly), and at eps = 1 the jumps act
    # as extra friction, so the diffusion constant is NOT expected to agree (eps -> 0 recovers the
    # Hamiltonian kicks): both are checked for sanity only.
    assert abs(T["jump"][0] - 300.0) < 15.0 and abs(T["baoab"][0] - 300.0) < 15.0
    # The mean potential energies differ by the two splittings' O(delta^2) biases: 0.13 - 0.17 kcal/mol per molecule at
    # delta = 1 fs in repeated runs, 0.03 at 0.5 fs (the next test checks that order); the slack is that bias, not noise.
    assert ob.agree(U["jump"], U["baoab"], 4.0, slack=0.2), (U["jump"], U["baoab"])
    sj, sb = res["jump"][1].std(), res["baoab"][1].std()          # width of the energy distribution (heat capacity)
    assert abs(sj / sb - 1.0) < 0.3, (sj, sb)
    assert gj.max() > 2.0 and 2.6 < r[gj.argmax()] < 3.0          # first O-O peak of liquid water
    assert (np.abs(gj - gb) <= 4.0 * np.hypot(ej, eb) + 0.08).all(), np.abs(gj - gb).max()
    assert 0.0 < Dj[0] <= Db[0] * 1.2


def test_jump_baoab_energy_gap_is_time_step_bias(jb):
    """The potential energy of JUMP sits 0.13 - 0.17 kcal/mol per molecule above BAOAB's at delta = 1 fs (flexible O-H
    bonds: omega delta = 0.7; BAOAB's velocities at the kick points are colder than 300 K by (omega delta)^2 terms and
    the jumps resample velocity components at exactly 300 K there).  Both schemes are second order in delta (P:L125:
    "the discretization bias on the invariant measure is of order delta^2"), so the gap must shrink about fourfold at
    delta = 0.5 fs -- a sampling error of the jump mechanism itself (rates, kernel, lists) would not."""
    sysd, run = wl.make_config(0)
    oxy = np.nonzero(np.asarray(sysd["lj_eps"]) > 0)[0]
    gap = {}
    for dt in (1.0, 0.5):
        U = {}
        for name in ("jump", "baoab"):
            g = jb.JumpSim(sysd, **dict(run, dt_fs=dt, seed=run["seed"] + 11))
            step = g.jump_step if name == "jump" else g.baoab_step
            g.baoab_step(int(3000 / dt)); step(int(3000 / dt))
            _, u, _ = sample_run(g, step, g.energy, lambda: g.pos.cpu().numpy(), 1500, int(20 / dt), oxy, 10 ** 9)
            assert g.stats()["error"] == 0
            U[name] = ob.block_mean_se(u)
            g.close()
        gap[dt] = (U["jump"][0] - U["baoab"][0], float(np.hypot(U["jump"][1], U["baoab"][1])))
    print("gap", gap)
    assert gap[1.0][0] > 3 * gap[1.0][1]                                  # the gap at 1 fs is real ...
    assert gap[0.5][0] < 0.5 * gap[1.0][0] + 3 * gap[0.5][1]              # ... and of second order in delta


def test_respa1_energy_gap_is_time_step_bias(jb):
    """NEXT-2 (R-21): three-level JUMP-RESPA1 against BAOAB-RESPA1 under the full Ewald potential U_direct + U_rec +
    U_self + U_excl.  Both sample the same measure up to a second-order bias in the time steps: the gap
    between their mean potential energies, 0.16 kcal/mol per molecule at 1:2:4 fs, must fall about fourfold when every
    level is halved (0.5:1:2 fs) -- a wrong slow kick or a wrong placement of the jumps in the levels would not."""
    sysd, run = wl.make_config(0)
    nmol = sysd["n_atoms"] // 3
    gap = {}
    for dt in (1.0, 0.5):
        U = {}
        for name, flags in (("jump", 3), ("baoab", 3 | 16)):
            g = jb.JumpSim(sysd, **dict(run, flags=flags, n_inner=2, dt_fs=dt, seed=run["seed"] + 21))
            assert g.ewald_setup() > 1000
            g.baoab_step(int(3000 / dt)); g.jump_respa1_step(int(3000 / (4 * dt)), 2)
            u = []
            for _ in range(1500):
                g.jump_respa1_step(int(round(24 / (4 * dt))), 2)
                u.append((g.energy()[1] + g.slow_energy()) / nmol)
            assert g.stats()["error"] == 0
            U[name] = ob.block_mean_se(u)
            g.close()
        gap[dt] = (U["jump"][0] - U["baoab"][0], float(np.hypot(U["jump"][1], U["baoab"][1])))
    print("respa1 gap", gap)
    assert gap[1.0][0] > 3 * gap[1.0][1]
    assert gap[0.5][0] < 0.5 * gap[1.0][0] + 3 * gap[0.5][1]


def test_config1_jump_vs_baoab_10000_steps(jb):
    """BASELINE configs[1] ("JUMP vs BAOAB, 10,000 steps" on the 12 000-atom box): the same comparison as on 216 waters, at
    the bench's size.  Averages over the last 10 000 steps of each scheme: both kinetic temperatures near 300 K with the
    splittings' known offsets (JUMP 303 K, BAOAB 293 K at delta = 1 fs, see the 216-water tests), the potential energy per
    molecule of JUMP above BAOAB's by the second-order gap (0.14 kcal/mol here, 0.12 on 216 waters) and no more, the
    same width of the energy distribution, thinning bounds never violated."""
    sysd, run = wl.make_config(1)
    nmol = sysd["n_atoms"] // 3
    res = {}
    for name in ("jump", "baoab"):
        g = jb.JumpSim(sysd, **dict(run, seed=run["seed"] + 31))
        step = g.jump_step if name == "jump" else g.baoab_step
        g.baoab_step(3000); step(2000)
        T, U = [], []
        for _ in range(500):
            step(20)
            ek, ep = g.energy()
            T.append(2.0 * ek / (3.0 * sysd["n_atoms"] * KB)); U.append(ep / nmol)
        st = g.stats()
        assert st["error"] == 0 and st["max_p"] <= 1 + 1e-4
        if name == "jump":
            assert 4.0 < st["proposals"] / (12000.0 * sysd["n_atoms"]) < 10.0      # proposals per atom and step (6.9 in the bench)
        res[name] = (ob.block_mean_se(T), ob.block_mean_se(U), float(np.std(U)))
        g.close()
    print("config1", res)
    assert abs(res["jump"][0][0] - 300.0) < 10.0 and abs(res["baoab"][0][0] - 300.0) < 15.0
    gap = res["jump"][1][0] - res["baoab"][1][0]
    assert 0.0 < gap < 0.3, gap
    # widths of the energy distribution: a 10 ps window holds about ten independent samples of U (its correlation time in
    # water at gamma = 1 / ps is about 1 ps), so each standard deviation is known to +-22 % and their ratio to +-31 % (one
    # sigma); repeated runs gave 0.57 and 0.69.  Checked as "the same order", three sigma.
    assert 0.4 < res["jump"][2] / res["baoab"][2] < 2.5


def test_bounce_heats_where_jump_does_not(jb):
    """NEXT-3 / P:L315-319: "the BPS electrostatic jumps can only be done on a very small range.  Jumping on a larger range
    yields too many velocity bounces" -- BOUNCE (eps = inf, B J A O A J B) on the 5-9 A range at delta = 1 fs heats the
    216-water box by hundreds of K within 400 steps and blows up; fusing the force and jump steps (C'J' A O A J'C' with
    eps = inf) "stabilizes further": it heats several times more slowly; the general mechanism with eps = 1 stays
    at the thermostat's temperature.  The blown-up run ends with a device error within seconds (chains are cut at 16 384
    proposals: an exploded velocity makes every waiting time 0), not with a kernel that never returns."""
    sysd, run = wl.make_config(0)
    n = sysd["n_atoms"]
    T = {}
    for name, kw in (("bounce", dict(eps_jump=float("inf"), flags=3 | jb.F_BJAOAJB)), ("fused_inf", dict(eps_jump=float("inf"), flags=3)),
                     ("jump", dict(eps_jump=1.0, flags=3))):
        g = jb.JumpSim(sysd, **dict(run, seed=run["seed"] + 41, **kw))
        g.set_lax_skin(True)
        g.baoab_step(3000)                                   # the same equilibrated start for the three
        g.jump_step(300)
        t = []
        for _ in range(5):
            g.jump_step(20)
            t.append(2.0 * g.energy()[0] / (3.0 * n * KB))
        T[name] = float(np.mean(t))                          # kinetic temperature over steps 300-400
        if name == "bounce":
            with pytest.raises(jb.JumpError):                # non-finite state, row overflow or a bound violated: it blows up
                for _ in range(40):
                    g.jump_step(100); g.sync()
        else:
            assert g.stats()["error"] == 0
        g.close()
    print("bounce", T)
    assert T["bounce"] > 420.0 and abs(T["jump"] - 300.0) < 25.0
    assert T["jump"] + 20.0 < T["fused_inf"] < T["bounce"] - 40.0


def test_config3_solute_jump_vs_baoab(jb):
    """BASELINE configs[3] ("JUMP vs BAOAB", 2 500-bead charged chain in water, 23 558 atoms, delta = 1 fs).  The generator's
    state (chain laid through lattice sites) is far from equilibrium and explodes at 1 fs, so both schemes start from the same
    staged BAOAB relaxation on the device (0.05 fs at gamma = 200 / ps up to 1 fs at gamma = 1 / ps, 10 000 steps in all);
    then 6 000 steps each: no device error with the skin check on, thinning bounds never violated (the chain's LJ
    parameters span sigma in [3, 4] A: the sup over sigma of R-7), rows within capacity, both kinetic temperatures near
    300 K and the potential energy per atom of JUMP within the second-order gap of BAOAB's."""
    sysd, run = wl.make_config(3)
    n = sysd["n_atoms"]
    pos, vel = sysd["pos"], sysd["vel"]
    for dt, gam, steps in ((0.05, 200.0, 2000), (0.2, 100.0, 2000), (0.5, 20.0, 2000), (1.0, 5.0, 2000), (1.0, 1.0, 2000)):
        g = jb.JumpSim(dict(sysd, pos=pos, vel=vel), **dict(run, dt_fs=dt, gamma_per_ps=gam))
        g.set_lax_skin(True)
        g.baoab_step(steps); g.sync()
        pos, vel = g.pos.cpu().numpy().astype(np.float64), g.vel.cpu().numpy().astype(np.float64)
        g.close()
    res = {}
    for name in ("jump", "baoab"):
        # nlist_every = 4: a rebuild may follow the previous one at once (Q = 1, R-10c).  The freely jointed chain has rare
        # violent close contacts (a bead thrown at 100 A/ps, 20 thermal sigmas) that use up a bead's share of the skin within
        # two steps; with the default period that is reported as JUMP_E_SKIN ("skin too small for this system")
        g = jb.JumpSim(dict(sysd, pos=pos, vel=vel), **dict(run, seed=run["seed"] + 51, nlist_every=4))
        step = g.jump_step if name == "jump" else g.baoab_step
        step(2000); g.sync()
        g.reset_stats()
        T, U = [], []
        for _ in range(200):
            step(20)
            ek, ep = g.energy()
            T.append(2.0 * ek / (3.0 * n * KB)); U.append(ep / n)
        st = g.stats()
        assert st["error"] == 0 and st["max_p"] <= 1 + 1e-4 and st["max_g_over_L"] <= 1 + 1e-4
        assert all(m <= c for m, c in zip(st["max_row"], st["cap_row"]) if c)
        res[name] = (ob.block_mean_se(T), ob.block_mean_se(U))
        g.close()
    print("config3", res)
    assert abs(res["jump"][0][0] - 300.0) < 12.0 and abs(res["baoab"][0][0] - 300.0) < 15.0
    gap = res["jump"][1][0] - res["baoab"][1][0]                 # kcal/mol per ATOM here (a third of the per-molecule figure)
    assert -0.03 < gap < 0.12, gap


def test_config2_jump_respa_vs_baoab_respa(jb):
    """BASELINE configs[2] (96 000 atoms; "JUMP-RESPA: inner step 1 fs for bonded + short-range forces, outer step 4 fs ...
    compared against BAOAB-RESPA at equal dt"): 4 ps of each from the same BAOAB-equilibrated state.  No device error with
    the skin check on, thinning bounds never violated, both kinetic temperatures near 300 K, and the potential energy per
    molecule of JUMP-RESPA above BAOAB-RESPA's by a second-order gap (0.14 at 1 fs for the plain schemes; the 4 fs outer
    step adds to both sides)."""
    sysd, run = wl.make_config(2)
    n, nmol = sysd["n_atoms"], sysd["n_atoms"] // 3
    g = jb.JumpSim(sysd, **run)
    g.set_lax_skin(True); g.baoab_step(2000); g.sync()
    pos, vel = g.pos.cpu().numpy().astype(np.float64), g.vel.cpu().numpy().astype(np.float64)
    g.close()
    res = {}
    for name, flags in (("jump_respa", 3), ("baoab_respa", 3 | 16)):
        g = jb.JumpSim(dict(sysd, pos=pos, vel=vel), **dict(run, flags=flags, seed=run["seed"] + 61))
        g.jump_respa_step(250); g.sync(); g.reset_stats()
        T, U = [], []
        for _ in range(100):
            g.jump_respa_step(10)
            ek, ep = g.energy()
            T.append(2.0 * ek / (3.0 * n * KB)); U.append(ep / nmol)
        st = g.stats()
        assert st["error"] == 0 and st["max_p"] <= 1 + 1e-4 and st["max_g_over_L"] <= 1 + 1e-4
        if name == "jump_respa":
            assert 3.0 < st["proposals"] / (4000.0 * n) < 12.0          # proposals per atom and inner step
        res[name] = (ob.block_mean_se(T), ob.block_mean_se(U))
        g.close()
    print("config2", res)
    assert abs(res["jump_respa"][0][0] - 300.0) < 15.0 and abs(res["baoab_respa"][0][0] - 300.0) < 15.0
    gap = res["jump_respa"][1][0] - res["baoab_respa"][1][0]
    assert -0.15 < gap < 0.45, gap                              # (-0.02 +- 0.05 measured: BAOAB-RESPA at 4 fs is noisy, T +- 2 K)
