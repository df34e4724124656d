"""ctypes front-end of the fp64 CPU oracle (oracle/jump_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT CODE: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It
imports nothing from the CUDA package and the CUDA package imports nothing
from here.  Every function is a thin call into the C file, which cites the
paper passage it follows.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "jump_oracle.c")
_LIB = os.path.join(_HERE, "libjump_oracle.so")

F_COUL_JUMPS, F_LJ_JUMPS, F_EVENT_LOG, F_RESPA_PAPER, F_RESPA_COMPARATOR = 1, 2, 4, 8, 16
F_BJAOAJB = 64
F_COMBINED = 128   # one mechanism per pair for the whole long pair gradient in (C'), no (J') (R-22)


def build(force=False):
    """Compile the oracle with gcc (-O2, OpenMP).  Building the checker is not using it."""
    if (not force) and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC):
        return _LIB
    tmp = _LIB + ".tmp%d" % os.getpid()
    cmd = ["gcc", "-O2", "-std=gnu99", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"]
    subprocess.check_call(cmd)
    os.replace(tmp, _LIB)
    return _LIB


class Params(C.Structure):
    _fields_ = [
        ("n_atoms", C.c_int32), ("n_inner", C.c_int32), ("eps_mode", C.c_int32), ("flags", C.c_uint32),
        ("nlist_every", C.c_int32), ("list_policy", C.c_int32), ("seed", C.c_uint64),
        ("box", C.c_double * 3),
        ("r_short", C.c_double), ("r_switch", C.c_double), ("r_mid", C.c_double), ("r_long", C.c_double),
        ("ewald_alpha", C.c_double),
        ("dt_fs", C.c_double), ("gamma_per_ps", C.c_double), ("temperature_K", C.c_double),
        ("eps_jump", C.c_double), ("skin", C.c_double), ("cell_edge", C.c_double), ("r_mid_in", C.c_double),
    ]


class Event(C.Structure):
    _fields_ = [
        ("step", C.c_int32), ("stream", C.c_int32), ("atom", C.c_int32), ("iter", C.c_int32),
        ("ring", C.c_int32), ("j", C.c_int32), ("accepted", C.c_int32), ("n_gt", C.c_int32),
        ("T", C.c_double), ("p", C.c_double), ("U", C.c_double), ("gt", C.c_double), ("margin", C.c_double),
    ]


EVENT_DTYPE = np.dtype([
    ("step", "i4"), ("stream", "i4"), ("atom", "i4"), ("iter", "i4"), ("ring", "i4"), ("j", "i4"),
    ("accepted", "i4"), ("n_gt", "i4"), ("T", "f8"), ("p", "f8"), ("U", "f8"), ("gt", "f8"), ("margin", "f8"),
])


class Stats(C.Structure):
    _fields_ = [
        ("proposals", C.c_int64), ("accepts", C.c_int64), ("gt_attempts", C.c_int64), ("rebuilds", C.c_int64),
        ("expiries", C.c_int64),
        ("max_p", C.c_double), ("max_g_over_L", C.c_double), ("max_disp", C.c_double), ("min_margin", C.c_double),
        ("min_margin_step", C.c_int64), ("min_list_margin", C.c_double), ("min_list_margin_step", C.c_int64),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int)
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.POINTER(Params), dp, dp, dp, dp, dp, dp, C.c_int, ip, dp, dp, C.c_int, ip, dp, dp, ip, ip]
        L.orc_free.argtypes = [C.c_void_p]
        for name in ("orc_jump_step", "orc_baoab_step", "orc_jump_respa_step"):
            getattr(L, name).argtypes = [C.c_void_p, C.c_int]
        L.orc_forces.argtypes = [C.c_void_p, C.c_int, C.c_int, dp]
        L.orc_potential.argtypes = [C.c_void_p, C.c_int]
        L.orc_potential.restype = C.c_double
        L.orc_kinetic.argtypes = [C.c_void_p]
        L.orc_kinetic.restype = C.c_double
        L.orc_get_state.argtypes = [C.c_void_p, C.c_int, dp]
        L.orc_set_state.argtypes = [C.c_void_p, dp, dp, C.c_int]
        L.orc_set_vel.argtypes = [C.c_void_p, dp]
        L.orc_get_events.argtypes = [C.c_void_p, C.c_void_p, C.c_int64]
        L.orc_get_events.restype = C.c_int64
        L.orc_clear_events.argtypes = [C.c_void_p]
        L.orc_get_stats.argtypes = [C.c_void_p, C.POINTER(Stats)]
        L.orc_reset_stats.argtypes = [C.c_void_p]
        L.orc_get_bounds.argtypes = [C.c_void_p, dp]
        L.orc_get_row_counts.argtypes = [C.c_void_p, ip, ip, ip]
        L.orc_get_row.argtypes = [C.c_void_p, C.c_int, C.c_int, ip, C.c_int]
        L.orc_get_row.restype = C.c_int
        L.orc_neighbors.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_int, C.c_int, ip, ip, C.c_int]
        L.orc_neighbors.restype = C.c_int
        L.orc_get_step.argtypes = [C.c_void_p]
        L.orc_get_step.restype = C.c_int64
        L.orc_set_eps.argtypes = [C.c_void_p, C.c_double]
        L.orc_scale_bounds.argtypes = [C.c_void_p, C.c_double]
        L.orc_set_bound_mode.argtypes = [C.c_void_p, C.c_int]
        L.orc_jump_half.argtypes = [C.c_void_p, C.c_double, C.c_int, C.c_int64]
        L.orc_ewald_setup.argtypes = [C.c_void_p, C.c_double]
        L.orc_ewald_nk.argtypes = [C.c_void_p]
        L.orc_ewald_nk.restype = C.c_int
        L.orc_jump_respa1_step.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.orc_fij.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, dp]
        L.orc_fij.restype = C.c_double
        L.orc_num_threads.restype = C.c_int
        # stand-alone functions (pins)
        L.orc_philox4x32_10.argtypes = [C.POINTER(C.c_uint32), C.POINTER(C.c_uint32), C.POINTER(C.c_uint32)]
        L.orc_u01.argtypes = [C.c_uint32]
        L.orc_u01.restype = C.c_double
        L.orc_chi.argtypes = [C.c_double, C.c_double, C.c_double, dp, dp]
        L.orc_u_coul.argtypes = [C.c_double, C.c_double, C.c_double, dp, dp]
        L.orc_u_lj.argtypes = [C.c_double, C.c_double, C.c_double, dp, dp]
        L.orc_weighted_du.argtypes = [C.c_int] + [C.c_double] * 6
        L.orc_weighted_du.restype = C.c_double
        L.orc_weighted_u.argtypes = [C.c_int] + [C.c_double] * 5
        L.orc_weighted_u.restype = C.c_double
        L.orc_theta.argtypes = [C.c_double]
        L.orc_theta.restype = C.c_double
        L.orc_jump_rate.argtypes = [C.c_double] * 5
        L.orc_jump_rate.restype = C.c_double
        L.orc_jump_kick.argtypes = [C.c_double, C.c_double, dp, C.c_double, dp]
        L.orc_gtilde_draw.argtypes = [C.c_double, C.c_uint64, C.c_int, C.c_int64, C.POINTER(C.c_int)]
        L.orc_gtilde_draw.restype = C.c_double
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int))


def make_params(n_atoms, box, r_short, r_long, r_switch=0.5, r_mid=None, ewald_alpha=-1.0, dt_fs=1.0,
                gamma_per_ps=1.0, temperature_K=300.0, n_inner=4, eps_jump=1.0, eps_mode=0,
                flags=F_COUL_JUMPS | F_LJ_JUMPS, skin=1.0, nlist_every=24, seed=0, cell_edge=0.0, list_policy=1,
                r_mid_in=None, **_ignored):
    """list_policy 1 (default, the contract of the CUDA path): DESIGN.md R-10c; 0: the ring rows of R-10."""
    p = Params()
    p.n_atoms, p.n_inner, p.eps_mode, p.flags = int(n_atoms), int(n_inner), int(eps_mode), int(flags)
    p.nlist_every, p.seed, p.list_policy = int(nlist_every), int(seed), int(list_policy)
    b = np.broadcast_to(np.asarray(box, dtype=np.float64), (3,))
    p.box[0], p.box[1], p.box[2] = float(b[0]), float(b[1]), float(b[2])
    p.r_short, p.r_switch, p.r_long = float(r_short), float(r_switch), float(r_long)
    p.r_mid = float(r_short + 2.0 if r_mid is None else r_mid)
    r_mid_in = r_short + 0.25 if r_mid_in is None else r_mid_in
    p.ewald_alpha = float(ewald_alpha)
    p.dt_fs, p.gamma_per_ps, p.temperature_K = float(dt_fs), float(gamma_per_ps), float(temperature_K)
    p.eps_jump, p.skin, p.cell_edge, p.r_mid_in = float(eps_jump), float(skin), float(cell_edge), float(r_mid_in)
    return p


class Oracle:
    """One oracle context.  `system` is a dict of numpy arrays as produced by the workload
    generator: pos, vel, mass, charge, lj_sigma, lj_eps, bond_ij, bond_k, bond_r0, angle_ijk,
    angle_k, angle_t0, excl_ptr, excl_idx (original atom indices throughout)."""

    def __init__(self, system, **params):
        L = lib()
        self.n = int(system["pos"].shape[0])
        kw = dict(params)
        kw.setdefault("box", system["box"])
        self.params = make_params(self.n, **kw)
        f8 = lambda k: np.ascontiguousarray(system[k], dtype=np.float64)
        i4 = lambda k: np.ascontiguousarray(system[k], dtype=np.int32)
        self._keep = [f8("pos"), f8("vel"), f8("mass"), f8("charge"), f8("lj_sigma"), f8("lj_eps"),
                      i4("bond_ij"), f8("bond_k"), f8("bond_r0"), i4("angle_ijk"), f8("angle_k"), f8("angle_t0"),
                      i4("excl_ptr"), i4("excl_idx")]
        k = self._keep
        self._h = L.orc_create(C.byref(self.params), _dp(k[0]), _dp(k[1]), _dp(k[2]), _dp(k[3]), _dp(k[4]), _dp(k[5]),
                               int(k[6].shape[0]), _ip(k[6]), _dp(k[7]), _dp(k[8]),
                               int(k[9].shape[0]), _ip(k[9]), _dp(k[10]), _dp(k[11]), _ip(k[12]), _ip(k[13]))

    def close(self):
        if self._h:
            lib().orc_free(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # --- stepping -----------------------------------------------------
    def jump_step(self, n=1):
        lib().orc_jump_step(self._h, int(n))

    def baoab_step(self, n=1):
        lib().orc_baoab_step(self._h, int(n))

    def jump_respa_step(self, n=1):
        lib().orc_jump_respa_step(self._h, int(n))

    def ewald_setup(self, k_cut=0.0):
        """Reciprocal vectors |k| <= k_cut (default 8 alpha) of the slow force of JUMP-RESPA1 (R-21); returns their number."""
        lib().orc_ewald_setup(self._h, float(k_cut))
        return lib().orc_ewald_nk(self._h)

    def jump_respa1_step(self, n=1, n_mid=3):
        """Three-level JUMP-RESPA1 / BAOAB-RESPA1: Delta = n_mid * n_inner * dt."""
        lib().orc_jump_respa1_step(self._h, int(n), int(n_mid))

    def jump_half(self, H_ps, with_accel=True, step=0):
        lib().orc_jump_half(self._h, float(H_ps), int(bool(with_accel)), int(step))

    # --- state --------------------------------------------------------
    def _state(self, which):
        out = np.empty((self.n, 3), dtype=np.float64)
        lib().orc_get_state(self._h, which, _dp(out))
        return out

    @property
    def pos(self):
        return self._state(0)

    @property
    def vel(self):
        return self._state(1)

    @property
    def pos_unwrapped(self):
        return self._state(2)

    def set_state(self, pos=None, vel=None, rebuild=True):
        x = None if pos is None else np.ascontiguousarray(pos, dtype=np.float64)
        v = None if vel is None else np.ascontiguousarray(vel, dtype=np.float64)
        lib().orc_set_state(self._h, None if x is None else _dp(x), None if v is None else _dp(v), int(bool(rebuild)))

    def set_vel(self, vel):
        v = np.ascontiguousarray(vel, dtype=np.float64)
        lib().orc_set_vel(self._h, _dp(v))

    @property
    def step(self):
        return int(lib().orc_get_step(self._h))

    # --- observables ----------------------------------------------------
    def forces(self, which=0, brute=False):
        """Gradient pieces in kcal/mol/A.  which: 0 F0, 1 full (unsplit to r_long), 2 long, 3 bonded, 4 short non-bonded."""
        out = np.empty((self.n, 3), dtype=np.float64)
        lib().orc_forces(self._h, int(which), int(bool(brute)), _dp(out))
        return out

    def potential(self, which=1):
        return float(lib().orc_potential(self._h, int(which)))

    def kinetic(self):
        return float(lib().orc_kinetic(self._h))

    def temperature(self):
        return 2.0 * self.kinetic() / (3.0 * self.n * 1.987204259e-3)

    def events(self):
        n = lib().orc_get_events(self._h, None, 0)
        buf = np.zeros(int(n), dtype=EVENT_DTYPE)
        assert buf.itemsize == C.sizeof(Event)
        if n:
            lib().orc_get_events(self._h, buf.ctypes.data_as(C.c_void_p), int(n))
        return buf

    def clear_events(self):
        lib().orc_clear_events(self._h)

    def stats(self):
        s = Stats()
        lib().orc_get_stats(self._h, C.byref(s))
        return {k: getattr(s, k) for k, _ in Stats._fields_}

    def reset_stats(self):
        lib().orc_reset_stats(self._h)

    def bounds(self):
        out = np.empty(12, dtype=np.float64)
        lib().orc_get_bounds(self._h, _dp(out))
        return dict(zip(["GM", "GL", "GV", "qmax", "eps_max", "sig_min", "sig_max", "rM", "G3", "GV2", "GV3", "rA"], out.tolist()))

    def row_counts(self):
        a = [np.empty(self.n, dtype=np.int32) for _ in range(3)]
        lib().orc_get_row_counts(self._h, _ip(a[0]), _ip(a[1]), _ip(a[2]))
        return a

    def row(self, which, i):
        cap = self.n
        out = np.empty(cap, dtype=np.int32)
        m = lib().orc_get_row(self._h, int(which), int(i), _ip(out), cap)
        return out[:m].copy()

    def neighbors(self, rmin, rmax, lj_only=False, brute=False):
        ptr = np.empty(self.n + 1, dtype=np.int32)
        tot = lib().orc_neighbors(self._h, float(rmin), float(rmax), int(lj_only), int(brute), _ip(ptr), None, 0)
        idx = np.empty(max(tot, 1), dtype=np.int32)
        lib().orc_neighbors(self._h, float(rmin), float(rmax), int(lj_only), int(brute), _ip(ptr), _ip(idx), tot)
        return ptr, idx[:tot]

    def fij(self, which, i, j):
        out = np.empty(3, dtype=np.float64)
        g = lib().orc_fij(self._h, int(which), int(i), int(j), _dp(out))
        return g, out

    def set_eps(self, eps):
        lib().orc_set_eps(self._h, float(eps))

    def scale_bounds(self, f):
        lib().orc_scale_bounds(self._h, float(f))

    def set_bound_mode(self, every_proposal):
        """R-11: False = bound held between accepted jumps (default); True = Algorithm 4 as printed (every proposal)."""
        lib().orc_set_bound_mode(self._h, int(bool(every_proposal)))


# --- stand-alone functions used by the pins ---------------------------------
def philox(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) & 0xFFFFFFFF for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) & 0xFFFFFFFF for x in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def u01(w):
    return float(lib().orc_u01(int(w) & 0xFFFFFFFF))


def chi(r, rc, h):
    a, b = C.c_double(), C.c_double()
    lib().orc_chi(float(r), float(rc), float(h), C.byref(a), C.byref(b))
    return a.value, b.value


def u_coul(r, qq, alpha):
    a, b = C.c_double(), C.c_double()
    lib().orc_u_coul(float(r), float(qq), float(alpha), C.byref(a), C.byref(b))
    return a.value, b.value


def u_lj(r, sig, eps):
    a, b = C.c_double(), C.c_double()
    lib().orc_u_lj(float(r), float(sig), float(eps), C.byref(a), C.byref(b))
    return a.value, b.value


def weighted_du(mode, r, rc, h, rlong, u, du):
    return float(lib().orc_weighted_du(int(mode), float(r), float(rc), float(h), float(rlong), float(u), float(du)))


def weighted_u(mode, r, rc, h, rlong, u):
    return float(lib().orc_weighted_u(int(mode), float(r), float(rc), float(h), float(rlong), float(u)))


def theta(eta):
    return float(lib().orc_theta(float(eta)))


def jump_rate(eps, beta, sbm, g, vn):
    return float(lib().orc_jump_rate(float(eps), float(beta), float(sbm), float(g), float(vn)))


def jump_kick(eps, sbm, n, gt, v):
    n = np.ascontiguousarray(n, dtype=np.float64)
    v = np.array(v, dtype=np.float64)
    lib().orc_jump_kick(float(eps), float(sbm), _dp(n), float(gt), _dp(v))
    return v


def gtilde_draw(eta, seed, atom, step=0):
    att = C.c_int()
    g = lib().orc_gtilde_draw(float(eta), int(seed), int(atom), int(step), C.byref(att))
    return float(g), att.value


def num_threads():
    return int(lib().orc_num_threads())


def pair_histogram(pos, box, r_max, n_bins):
    """NEXT-4 oracle: number of unordered pairs of the given points whose minimum-image distance r (cubic periodic box,
    P:L325) is < r_max, per bin floor(r n_bins / r_max) -- the plain definition, O(N^2), fp64.  g(r) follows by
    dividing by 0.5 N (N-1) / V times the shell volumes (the radial distribution functions of P:L527-531)."""
    x = np.asarray(pos, dtype=np.float64)
    hist = np.zeros(n_bins, dtype=np.int64)
    for i in range(len(x) - 1):
        d = x[i + 1:] - x[i]
        d -= box * np.round(d / box)
        r = np.sqrt((d * d).sum(1))
        b = np.floor(r[r < r_max] * (n_bins / r_max)).astype(np.int64)
        hist += np.bincount(np.minimum(b, n_bins - 1), minlength=n_bins)
    return hist


def velocity_autocorrelation(v_origin, v_now, select=None):
    """NEXT-4 oracle: C = (1/N_sel) sum_{i in sel} v_i(t0) . v_i(t0 + tau), (A/ps)^2 -- the plain definition of the
    velocity autocorrelation behind the spectra of P:L529-531, L583-589, fp64."""
    a, b = np.asarray(v_origin, dtype=np.float64), np.asarray(v_now, dtype=np.float64)
    if select is not None:
        a, b = a[select], b[select]
    return float((a * b).sum(1).mean())


def mean_square_displacement(x_origin_unwrapped, x_now_unwrapped, select=None):
    """NEXT-4 oracle: MSD = (1/N_sel) sum_{i in sel} |x_i(t0 + tau) - x_i(t0)|^2, A^2, on UNWRAPPED positions -- the plain
    definition behind the diffusion constants D = lim MSD / (6 tau) of P:L527, L575-581, fp64."""
    a, b = np.asarray(x_origin_unwrapped, dtype=np.float64), np.asarray(x_now_unwrapped, dtype=np.float64)
    if select is not None:
        a, b = a[select], b[select]
    return float(((b - a) ** 2).sum(1).mean())


def vacf_spectrum(c, dt_ps, omegas):
    """I(omega) = dt [C(0)/2 + sum_{k>=1} C(k dt) cos(omega k dt) w_k] with a Hann window w_k = cos^2(pi k / 2K) over the K
    lags given: the windowed cosine transform of the autocorrelation (the velocity spectra of P:L529-531), fp64."""
    c = np.asarray(c, dtype=np.float64)
    k = np.arange(len(c))
    w = np.cos(0.5 * np.pi * k / len(c)) ** 2
    w[0] = 0.5
    return np.array([dt_ps * float((c * w * np.cos(om * k * dt_ps)).sum()) for om in np.atleast_1d(omegas)])
