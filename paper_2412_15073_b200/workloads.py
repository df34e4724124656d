"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json configs 0-4).

This module holds NONE of the method's arithmetic (no forces, no integrator, no
random-number contract): it only lays atoms out.  It is the one module that both
the tests of the fp64 oracle and the CUDA path (tests, bench.py, smoke) read
inputs from, and it imports neither of them.

The paper measured on Tinker-HP SPC/Fw water boxes (Table 4)
that are not available here; these boxes stand in for them with the same atom
counts, box sizes, charges and Lennard-Jones parameters ("Input
recipe").  All returned floats are exactly representable in fp32, so the fp32
CUDA path and the fp64 oracle start from bit-identical values.
"""
import numpy as np

KB = 1.987204259e-3  # kcal/mol/K
KCAL = 418.4         # (g/mol) A^2 ps^-2 per kcal/mol

WATER = dict(qO=-0.834, qH=0.417, sigma=3.1507, eps=0.1521, r0=0.9572, kb=450.0,
             theta0_deg=104.52, ka=55.0, mO=15.999, mH=1.008)

# BASELINE.json configs[k]; seeds per SURVEY 8(d): structure 1000+k, velocities 2000+k, dynamics 3000+k
CONFIGS = {
    0: dict(kind="water", n_mol=216, box=18.64, r_short=5.0, r_long=9.0, dt_fs=1.0, n_inner=4),
    1: dict(kind="water", n_mol=4000, box=49.3, r_short=6.0, r_long=12.0, dt_fs=1.0, n_inner=4),
    2: dict(kind="water", n_mol=32000, box=98.6, r_short=6.0, r_long=12.0, dt_fs=1.0, n_inner=4),
    3: dict(kind="solute", n_mol=7019, n_beads=2500, box=62.0, r_short=6.0, r_long=12.0, dt_fs=1.0, n_inner=4),
    4: dict(kind="water", n_mol=333333, box=215.2, r_short=6.0, r_long=12.0, dt_fs=1.0, n_inner=4),
}


def _f32(a):
    return np.asarray(a, dtype=np.float32).astype(np.float64)


def _random_rotations(rng, n):
    """n uniform random rotation matrices (from unit quaternions)."""
    q = rng.normal(size=(n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    R = np.empty((n, 3, 3))
    R[:, 0, 0] = 1 - 2 * (y * y + z * z); R[:, 0, 1] = 2 * (x * y - z * w); R[:, 0, 2] = 2 * (x * z + y * w)
    R[:, 1, 0] = 2 * (x * y + z * w); R[:, 1, 1] = 1 - 2 * (x * x + z * z); R[:, 1, 2] = 2 * (y * z - x * w)
    R[:, 2, 0] = 2 * (x * z - y * w); R[:, 2, 1] = 2 * (y * z + x * w); R[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return R


def _water_template():
    th = np.deg2rad(WATER["theta0_deg"])
    r0 = WATER["r0"]
    return np.array([[0.0, 0.0, 0.0],
                     [r0 * np.sin(th / 2), 0.0, r0 * np.cos(th / 2)],
                     [-r0 * np.sin(th / 2), 0.0, r0 * np.cos(th / 2)]])


def _place_waters(rng, sites_ijk, n_side, a, hh_min=1.8, tries=40):
    """Waters on lattice sites, uniformly random orientations; an orientation is redrawn while
    one of its H sits closer than hh_min to an H of an already placed neighbour (pure geometry:
    avoids the few very high-energy contacts of a blind random start)."""
    n = sites_ijk.shape[0]
    tmpl = _water_template()
    site_of = -np.ones((n_side, n_side, n_side), dtype=np.int64)
    site_of[sites_ijk[:, 0], sites_ijk[:, 1], sites_ijk[:, 2]] = np.arange(n)
    centre = (sites_ijk + 0.5) * a
    rel = np.zeros((n, 3, 3))          # atom offsets from the O site
    placed = np.zeros(n, dtype=bool)
    colour = (sites_ijk[:, 0] % 2) + 2 * (sites_ijk[:, 1] % 2) + 4 * (sites_ijk[:, 2] % 2)
    offs = np.array([(i, j, k) for i in (-1, 0, 1) for j in (-1, 0, 1) for k in (-1, 0, 1) if (i, j, k) != (0, 0, 0)])
    for col in range(8):
        todo = np.nonzero(colour == col)[0]
        for _ in range(tries):
            if todo.size == 0:
                break
            R = _random_rotations(rng, todo.size)
            cand = np.einsum("nij,aj->nai", R, tmpl)       # (m, 3 atoms, 3)
            ok = np.ones(todo.size, dtype=bool)
            for o in offs:
                nb_ijk = (sites_ijk[todo] + o) % n_side
                nb = site_of[nb_ijk[:, 0], nb_ijk[:, 1], nb_ijk[:, 2]]
                has = (nb >= 0) & placed[np.maximum(nb, 0)]
                if not has.any():
                    continue
                shift = o * a                               # neighbour centre relative to ours (lattice image)
                hn = rel[np.maximum(nb, 0)][:, 1:, :] + shift
                d = np.linalg.norm(cand[:, 1:, None, :] - hn[:, None, :, :], axis=-1)
                ok &= ~(has & (d.min(axis=(1, 2)) < hh_min))
            good = todo[ok]
            rel[good] = cand[ok]
            placed[good] = True
            todo = todo[~ok]
        if todo.size:                                       # keep the last draw for the few left over
            R = _random_rotations(rng, todo.size)
            rel[todo] = np.einsum("nij,aj->nai", R, tmpl)
            placed[todo] = True
    return centre[:, None, :] + rel


def _maxwell(rng, mass, temperature):
    sd = np.sqrt(KB * temperature * KCAL / mass)            # A/ps
    return rng.normal(size=(mass.shape[0], 3)) * sd[:, None]


def _csr_from_lists(lists):
    ptr = np.zeros(len(lists) + 1, dtype=np.int32)
    for i, l in enumerate(lists):
        ptr[i + 1] = ptr[i] + len(l)
    idx = np.array([j for l in lists for j in l], dtype=np.int32) if ptr[-1] else np.zeros(0, dtype=np.int32)
    return ptr, idx


def water_box(n_mol, box, seed_struct, seed_vel, temperature=300.0):
    """Flexible 3-site water (BASELINE.json configs 0, 1, 2, 4)."""
    rng = np.random.default_rng(seed_struct)
    box = float(np.float32(box))
    n_side = int(np.ceil(n_mol ** (1.0 / 3.0) - 1e-9))
    n_side += n_side % 2                                     # even, for the 8-colour placement
    a = box / n_side
    n_sites = n_side ** 3
    chosen = np.sort(rng.permutation(n_sites)[:n_mol]) if n_mol < n_sites else np.arange(n_sites)
    ijk = np.stack([chosen // (n_side * n_side), (chosen // n_side) % n_side, chosen % n_side], axis=1)
    xyz = _place_waters(rng, ijk, n_side, a)                # (n_mol, 3, 3)
    pos = _f32(np.mod(xyz.reshape(-1, 3), box))
    pos[pos >= box] = 0.0                                    # fp32 rounding may land exactly on the edge
    n = 3 * n_mol
    W = WATER
    mass = np.tile([W["mO"], W["mH"], W["mH"]], n_mol).astype(np.float64)
    charge = np.tile([W["qO"], W["qH"], W["qH"]], n_mol).astype(np.float64)
    lj_sigma = np.tile([W["sigma"], 1.0, 1.0], n_mol).astype(np.float64)
    lj_eps = np.tile([W["eps"], 0.0, 0.0], n_mol).astype(np.float64)
    o = 3 * np.arange(n_mol, dtype=np.int32)
    bond_ij = np.stack([np.repeat(o, 2), (o[:, None] + np.array([1, 2], dtype=np.int32)).ravel()], axis=1).astype(np.int32)
    bond_k = np.full(2 * n_mol, W["kb"])
    bond_r0 = np.full(2 * n_mol, W["r0"])
    angle_ijk = np.stack([o + 1, o, o + 2], axis=1).astype(np.int32)   # vertex in the middle
    angle_k = np.full(n_mol, W["ka"])
    angle_t0 = np.full(n_mol, np.deg2rad(W["theta0_deg"]))
    excl_ptr = (2 * np.arange(n + 1)).astype(np.int32)
    base = np.repeat(o, 3)
    within = np.tile(np.array([[1, 2], [0, 2], [0, 1]], dtype=np.int32), (n_mol, 1))
    excl_idx = (base[:, None] + within).ravel().astype(np.int32)
    vel = _maxwell(np.random.default_rng(seed_vel), mass, temperature)
    return dict(kind="water", n_atoms=n, box=float(np.float32(box)),
                pos=_f32(pos), vel=_f32(vel), mass=_f32(mass), charge=_f32(charge),
                lj_sigma=_f32(lj_sigma), lj_eps=_f32(lj_eps),
                bond_ij=bond_ij, bond_k=_f32(bond_k), bond_r0=_f32(bond_r0),
                angle_ijk=angle_ijk, angle_k=_f32(angle_k), angle_t0=_f32(angle_t0),
                excl_ptr=excl_ptr, excl_idx=excl_idx)


def solute_box(n_mol, n_beads, box, seed_struct, seed_vel, temperature=300.0):
    """Config 3 mimic: a charged bead chain folded along lattice sites inside a water box.
    23 558 = 2 500 beads + 7 019 waters (21 057 atoms) + 1 neutral free LJ bead."""
    rng = np.random.default_rng(seed_struct)
    n_side = int(np.ceil((n_mol + n_beads) ** (1.0 / 3.0) + 1.0))
    n_side += n_side % 2
    a = box / n_side
    # chain: a boustrophedon (snake) walk through a compact cube of sites -> consecutive beads are
    # lattice neighbours and no site is used twice.  The walk spacing a (~2.9 A) is longer than the
    # 1.53 A bond, so beads are pulled to the bond length along the path.
    m = int(np.ceil(n_beads ** (1.0 / 3.0)))
    path = []
    for k in range(m):
        for j in (range(m) if k % 2 == 0 else range(m - 1, -1, -1)):
            row = range(m) if (j + k * m) % 2 == 0 else range(m - 1, -1, -1)
            for i in row:
                path.append((i, j, k))
    path = np.array(path[:n_beads]) + (n_side - m) // 2
    used = np.zeros((n_side,) * 3, dtype=bool)
    used[path[:, 0], path[:, 1], path[:, 2]] = True
    # keep beads on their sites (spacing a): the harmonic bonds (r0 = 1.53 A) relax them in the
    # equilibration that every run starts with; sites next to the chain stay empty of water.
    bead_pos = (path + 0.5) * a
    free = np.argwhere(~used)
    # drop water sites that touch the chain (closer than one lattice spacing)
    near = np.zeros_like(used)
    for o in [(1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)]:
        near |= np.roll(used, o, axis=(0, 1, 2))
    free = np.array([s for s in free if not near[tuple(s)]])
    sel = np.sort(rng.permutation(free.shape[0])[: n_mol + 1])
    w_sites = free[sel[:n_mol]]
    extra_site = free[sel[n_mol]]
    xyz = _place_waters(rng, w_sites, n_side, a)
    W = WATER
    nb = n_beads
    q = rng.normal(0.0, 0.3, size=nb)
    q -= q.mean()
    sig = rng.uniform(3.0, 4.0, size=nb)
    eps = rng.uniform(0.05, 0.2, size=nb)
    nw = 3 * n_mol
    n = nb + nw + 1
    pos = np.concatenate([bead_pos, xyz.reshape(-1, 3), ((extra_site + 0.5) * a)[None, :]], axis=0)
    mass = np.concatenate([np.full(nb, 12.011), np.tile([W["mO"], W["mH"], W["mH"]], n_mol), [12.011]])
    charge = np.concatenate([q, np.tile([W["qO"], W["qH"], W["qH"]], n_mol), [0.0]])
    lj_sigma = np.concatenate([sig, np.tile([W["sigma"], 1.0, 1.0], n_mol), [3.5]])
    lj_eps = np.concatenate([eps, np.tile([W["eps"], 0.0, 0.0], n_mol), [0.1]])
    o = nb + 3 * np.arange(n_mol, dtype=np.int32)
    cb = np.stack([np.arange(nb - 1), np.arange(1, nb)], axis=1)
    wb = np.stack([np.repeat(o, 2), (o[:, None] + np.array([1, 2])).ravel()], axis=1)
    bond_ij = np.concatenate([cb, wb]).astype(np.int32)
    bond_k = np.concatenate([np.full(nb - 1, 300.0), np.full(2 * n_mol, W["kb"])])
    bond_r0 = np.concatenate([np.full(nb - 1, 1.53), np.full(2 * n_mol, W["r0"])])
    angle_ijk = np.stack([o + 1, o, o + 2], axis=1).astype(np.int32)
    angle_k = np.full(n_mol, W["ka"])
    angle_t0 = np.full(n_mol, np.deg2rad(W["theta0_deg"]))
    lists = [[] for _ in range(n)]
    for i in range(nb):                                     # 1-2 and 1-3 along the chain (R-9)
        for d in (-2, -1, 1, 2):
            if 0 <= i + d < nb:
                lists[i].append(i + d)
    for mol in range(n_mol):
        b = nb + 3 * mol
        lists[b] = [b + 1, b + 2]; lists[b + 1] = [b, b + 2]; lists[b + 2] = [b, b + 1]
    excl_ptr, excl_idx = _csr_from_lists(lists)
    vel = _maxwell(np.random.default_rng(seed_vel), mass, temperature)
    return dict(kind="solute", n_atoms=n, box=float(np.float32(box)),
                pos=_f32(np.mod(pos, box)), vel=_f32(vel), mass=_f32(mass), charge=_f32(charge),
                lj_sigma=_f32(lj_sigma), lj_eps=_f32(lj_eps),
                bond_ij=bond_ij, bond_k=_f32(bond_k), bond_r0=_f32(bond_r0),
                angle_ijk=angle_ijk, angle_k=_f32(angle_k), angle_t0=_f32(angle_t0),
                excl_ptr=excl_ptr, excl_idx=excl_idx)


def make_config(k, temperature=300.0):
    """(system dict, run-parameter dict) of BASELINE.json configs[k]."""
    cfg = CONFIGS[k]
    if cfg["kind"] == "water":
        sysd = water_box(cfg["n_mol"], cfg["box"], 1000 + k, 2000 + k, temperature)
    else:
        sysd = solute_box(cfg["n_mol"], cfg["n_beads"], cfg["box"], 1000 + k, 2000 + k, temperature)
    run = dict(r_short=cfg["r_short"], r_long=cfg["r_long"], r_switch=0.5, r_mid=cfg["r_short"] + 2.0,
               r_mid_in=cfg["r_short"] + 0.25,
               ewald_alpha=-1.0, dt_fs=cfg["dt_fs"], gamma_per_ps=1.0, temperature_K=temperature,
               n_inner=cfg["n_inner"], eps_jump=1.0, eps_mode=0, flags=3, skin=1.0, nlist_every=24,
               seed=3000 + k,
               # edge of the contract grid's cells (R-10c): the default rule, (r_long + skin w_max) / 4 = 3.3 A, on the 9 A box;
               # 4.7 A on the 12 A boxes (measured on the 10^6-atom box, 1 000-step runs: 3.3 A 48.8, 4.0 48.2, 4.4 50.1,
               # 4.5 49.0, 4.7 51.2, 5.0 50.6, 5.4 49.2 ns/day -- fewer, fuller cells for the list kernels against a larger
               # universe for ring C)
               cell_edge=0.0 if cfg["r_long"] < 10.0 else 4.7)
    return sysd, run


def small_water(n_side, seed=7, box=None, temperature=300.0):
    """A small water box (n_side^3 molecules at liquid density) for unit tests."""
    n_mol = n_side ** 3
    if box is None:
        box = (n_mol * 29.915) ** (1.0 / 3.0)
    return water_box(n_mol, box, seed, seed + 1, temperature)
