"""Thin ctypes binding of libjump_b200.so (include/jump_b200.h): argument marshalling only.

PyTorch is used for device memory and streams; every step of the path runs in the library's CUDA
kernels.  There is no CPU fallback: importing works without a GPU (so that the symbol check can
run), but creating a context without the built library or without a CUDA device raises.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libjump_b200.so")

F_COUL_JUMPS, F_LJ_JUMPS, F_EVENT_LOG, F_RESPA_PAPER, F_RESPA_COMPARATOR = 1, 2, 4, 8, 16
F_LAX_SKIN = 32
F_BJAOAJB = 64
F_COMBINED = 128
ERRORS = {-1: "bad argument", -2: "CUDA error", -3: "row/event overflow", -4: "thinning bound violated",
          -5: "displacement beyond skin/2", -6: "non-finite state"}

EXPORTS = ["jump_init", "jump_step", "baoab_step", "jump_respa_step", "jump_get_forces", "jump_get_energy",
           "jump_get_stats", "jump_reset_stats", "jump_get_events", "jump_clear_events", "jump_get_row", "jump_get_images", "jump_rdf_accumulate",
           "jump_get_bounds", "jump_refresh", "jump_refresh_lazy", "jump_half", "jump_sync", "jump_get_step", "jump_get_launches",
           "jump_last_error", "jump_free", "jump_set_profiling", "jump_get_profile", "jump_count_pairs",
           "jump_ewald_setup", "jump_respa1_step", "jump_get_slow_energy", "jump_vacf_mark", "jump_vacf_dot", "jump_msd_mark", "jump_msd", "jump_set_lanes", "jump_set_lax_skin",
           "jump_vacf_static_setup", "jump_vacf_dot_static", "jump_vacf_static_last_error"]


class jump_params(C.Structure):
    _fields_ = [
        ("n_atoms", C.c_int32), ("n_inner", C.c_int32), ("eps_mode", C.c_int32), ("flags", C.c_uint32),
        ("nlist_every", C.c_int32), ("pad0", C.c_int32), ("seed", C.c_uint64),
        ("box", C.c_double * 3),
        ("r_short", C.c_double), ("r_switch", C.c_double), ("r_mid", C.c_double), ("r_long", C.c_double),
        ("ewald_alpha", C.c_double),
        ("dt_fs", C.c_double), ("gamma_per_ps", C.c_double), ("temperature_K", C.c_double),
        ("eps_jump", C.c_double), ("skin", C.c_double), ("cell_edge", C.c_double), ("r_mid_in", C.c_double),
    ]


class jump_event(C.Structure):
    _fields_ = [("step", C.c_int32), ("stream", C.c_int32), ("atom", C.c_int32), ("iter", C.c_int32),
                ("ring", C.c_int32), ("j", C.c_int32), ("accepted", C.c_int32), ("n_gt", C.c_int32),
                ("T", C.c_float), ("p", C.c_float), ("U", C.c_float), ("gt", C.c_float)]


EVENT_DTYPE = np.dtype([("step", "i4"), ("stream", "i4"), ("atom", "i4"), ("iter", "i4"), ("ring", "i4"), ("j", "i4"),
                        ("accepted", "i4"), ("n_gt", "i4"), ("T", "f4"), ("p", "f4"), ("U", "f4"), ("gt", "f4")])


class jump_stats(C.Structure):
    _fields_ = [("proposals", C.c_int64), ("accepts", C.c_int64), ("gt_attempts", C.c_int64), ("rebuilds", C.c_int64),
                ("expiries", C.c_int64), ("max_p", C.c_double), ("max_g_over_L", C.c_double), ("max_disp", C.c_double),
                ("max_row", C.c_int32 * 6), ("cap_row", C.c_int32 * 6), ("error", C.c_int32), ("pad", C.c_int32)]


_lib = None


def build(force=False):
    from . import build as _b
    return _b.build(force=force)


def lib():
    """Load the C-ABI library (raises if it has not been built: there is no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libjump_b200.so is missing: run `python -m paper_2412_15073_b200.build` "
                               "(or __graft_entry__.build()); the CUDA path has no CPU fallback")
        L = C.CDLL(LIB_PATH)
        vp, i32, i64, dp = C.c_void_p, C.c_int32, C.c_int64, C.POINTER(C.c_double)
        L.jump_init.argtypes = [C.POINTER(vp), C.POINTER(jump_params), vp, vp, vp, vp, vp, vp, i32, vp, vp, vp, i32, vp, vp, vp,
                                vp, vp, vp]
        L.jump_step.argtypes = [vp, i32]
        L.baoab_step.argtypes = [vp, i32]
        L.jump_respa_step.argtypes = [vp, i32]
        L.jump_ewald_setup.argtypes = [vp, C.c_double, C.POINTER(C.c_int32)]
        L.jump_respa1_step.argtypes = [vp, i32, i32]
        L.jump_get_slow_energy.argtypes = [vp, C.POINTER(C.c_double)]
        L.jump_msd_mark.argtypes = [vp]
        L.jump_msd.argtypes = [vp, i32, C.POINTER(C.c_double)]
        L.jump_vacf_mark.argtypes = [vp]
        L.jump_vacf_dot.argtypes = [vp, i32, C.POINTER(C.c_double)]
        L.jump_get_forces.argtypes = [vp, i32, vp]
        L.jump_get_energy.argtypes = [vp, dp, dp]
        L.jump_get_stats.argtypes = [vp, C.POINTER(jump_stats)]
        L.jump_reset_stats.argtypes = [vp]
        L.jump_get_events.argtypes = [vp, vp, i64, C.POINTER(i64)]
        L.jump_clear_events.argtypes = [vp]
        L.jump_get_row.argtypes = [vp, i32, i32, C.POINTER(i32), i32]
        L.jump_get_bounds.argtypes = [vp, dp]
        L.jump_get_images.argtypes = [vp, vp]
        L.jump_rdf_accumulate.argtypes = [vp, i32, C.c_double, i32, vp]
        L.jump_refresh.argtypes = [vp]
        L.jump_refresh_lazy.argtypes = [vp, C.POINTER(i32)]
        L.jump_half.argtypes = [vp, C.c_double, i32, i64]
        L.jump_sync.argtypes = [vp]
        L.jump_get_step.argtypes = [vp]
        L.jump_get_step.restype = i64
        L.jump_get_launches.argtypes = [vp]
        L.jump_get_launches.restype = i64
        L.jump_last_error.argtypes = [vp]
        L.jump_last_error.restype = C.c_char_p
        L.jump_free.argtypes = [vp]
        L.jump_free.restype = None
        L.jump_set_profiling.argtypes = [vp, i32]
        L.jump_get_profile.argtypes = [vp, dp, C.POINTER(i64)]
        L.jump_count_pairs.argtypes = [vp, i32, C.c_double, C.POINTER(i64)]
        L.jump_set_lanes.argtypes = [vp, i32]
        L.jump_set_lax_skin.argtypes = [vp, i32]
        L.jump_vacf_static_setup.argtypes = []
        L.jump_vacf_dot_static.argtypes = [i32, vp, vp, vp, vp, vp]
        L.jump_vacf_static_last_error.argtypes = []
        L.jump_vacf_static_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def make_params(n_atoms, box, r_short, r_long, r_switch=0.5, r_mid=None, ewald_alpha=-1.0, dt_fs=1.0, gamma_per_ps=1.0,
                temperature_K=300.0, n_inner=4, eps_jump=1.0, eps_mode=0, flags=F_COUL_JUMPS | F_LJ_JUMPS, skin=1.0,
                nlist_every=24, seed=0, cell_edge=0.0, r_mid_in=None, **_ignored):
    p = jump_params()
    p.n_atoms, p.n_inner, p.eps_mode, p.flags = int(n_atoms), int(n_inner), int(eps_mode), int(flags)
    p.nlist_every, p.seed = int(nlist_every), int(seed)
    b = np.broadcast_to(np.asarray(box, dtype=np.float64), (3,))
    p.box[0], p.box[1], p.box[2] = float(b[0]), float(b[1]), float(b[2])
    p.r_short, p.r_switch, p.r_long = float(r_short), float(r_switch), float(r_long)
    p.r_mid = float(r_short + 2.0 if r_mid is None else r_mid)
    r_mid_in = r_short + 0.25 if r_mid_in is None else r_mid_in
    p.ewald_alpha = float(ewald_alpha)
    p.dt_fs, p.gamma_per_ps, p.temperature_K = float(dt_fs), float(gamma_per_ps), float(temperature_K)
    p.eps_jump, p.skin, p.cell_edge, p.r_mid_in = float(eps_jump), float(skin), float(cell_edge), float(r_mid_in)
    return p


class JumpError(RuntimeError):
    pass


VACF_STATIC_MAX_ATOMS = 4194304


def vacf_dot_static(v_now, v_origin, out, select=None, stream=None):
    """jump_vacf_dot_static: (1/N_sel) sum v_i(origin) . v_i(now) and N_sel into `out` (2 float64 on the device) with no
    allocation by the library (scratch in a static device array; at most VACF_STATIC_MAX_ATOMS atoms).  v_now,
    v_origin: contiguous (n, 3) float32 CUDA tensors; select: (n,) int32 or None.  Asynchronous on `stream`."""
    import torch
    for t in (v_now, v_origin):
        assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and t.dim() == 2 and t.shape[1] == 3
    assert v_now.shape == v_origin.shape and out.is_cuda and out.dtype == torch.float64 and out.numel() == 2 and out.is_contiguous()
    if select is not None:
        assert select.is_cuda and select.dtype == torch.int32 and select.is_contiguous() and select.numel() == v_now.shape[0]
    st = stream if stream is not None else torch.cuda.current_stream(v_now.device)
    L = lib()
    with torch.cuda.device(v_now.device):
        rc = L.jump_vacf_dot_static(int(v_now.shape[0]), C.c_void_p(v_now.data_ptr()), C.c_void_p(v_origin.data_ptr()),
                                    C.c_void_p(select.data_ptr() if select is not None else 0), C.c_void_p(out.data_ptr()),
                                    C.c_void_p(st.cuda_stream))
    if rc < 0:
        raise JumpError("jump_vacf_dot_static failed: %d (%s) %s" % (rc, ERRORS.get(rc, "?"),
                                                                     (L.jump_vacf_static_last_error() or b"").decode()))
    return out


class JumpSim:
    """One simulation context on the current CUDA device.  `system` is a dict of numpy arrays as made by
    paper_2412_15073_b200.workloads (original atom indices throughout); run parameters as keywords."""

    def __init__(self, system, device="cuda:0", stream=None, **params):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2412_15073_b200 needs a CUDA device: there is no CPU fallback")
        self._torch = torch
        self._L = lib()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.n = int(system["pos"].shape[0])
        kw = dict(params)
        kw.setdefault("box", system["box"])
        self.params = make_params(self.n, **kw)
        f32 = lambda k: torch.as_tensor(np.ascontiguousarray(system[k], dtype=np.float32), device=self.device)
        i32 = lambda k: torch.as_tensor(np.ascontiguousarray(system[k], dtype=np.int32), device=self.device)
        self.pos, self.vel = f32("pos"), f32("vel")          # updated in place by the library
        self._keep = [f32("mass"), f32("charge"), f32("lj_sigma"), f32("lj_eps"), i32("bond_ij"), f32("bond_k"),
                      f32("bond_r0"), i32("angle_ijk"), f32("angle_k"), f32("angle_t0"), i32("excl_ptr"), i32("excl_idx")]
        k = self._keep
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        h = C.c_void_p()
        ptr = lambda t: C.c_void_p(t.data_ptr()) if t.numel() else C.c_void_p(0)
        torch.cuda.synchronize(self.device)
        rc = self._L.jump_init(C.byref(h), C.byref(self.params), ptr(self.pos), ptr(self.vel), ptr(k[0]), ptr(k[1]), ptr(k[2]),
                               ptr(k[3]), int(k[4].shape[0]), ptr(k[4]), ptr(k[5]), ptr(k[6]), int(k[7].shape[0]), ptr(k[7]),
                               ptr(k[8]), ptr(k[9]), ptr(k[10]), ptr(k[11]), C.c_void_p(self.stream.cuda_stream))
        self._h = h
        self._check(rc, "jump_init")

    def _check(self, rc, what):
        if rc < 0:
            msg = self._L.jump_last_error(self._h) if self._h else b""
            raise JumpError("%s failed: %d (%s) %s" % (what, rc, ERRORS.get(rc, "?"), (msg or b"").decode()))
        return rc

    def close(self):
        if getattr(self, "_h", None):
            self._L.jump_free(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the hot path (asynchronous; same names as the C entry points) -------------------------------
    def jump_step(self, n=1):
        self._check(self._L.jump_step(self._h, int(n)), "jump_step")

    def baoab_step(self, n=1):
        self._check(self._L.baoab_step(self._h, int(n)), "baoab_step")

    def jump_respa_step(self, n=1):
        self._check(self._L.jump_respa_step(self._h, int(n)), "jump_respa_step")

    def ewald_setup(self, k_cut=0.0):
        """Reciprocal vectors |k| <= k_cut (default 8 alpha) of the slow force of JUMP-RESPA1; returns their number."""
        nk = C.c_int32(0)
        self._check(self._L.jump_ewald_setup(self._h, float(k_cut), C.byref(nk)), "jump_ewald_setup")
        return int(nk.value)

    def jump_respa1_step(self, n=1, n_mid=3):
        self._check(self._L.jump_respa1_step(self._h, int(n), int(n_mid)), "jump_respa1_step")

    def msd_mark(self):
        self._check(self._L.jump_msd_mark(self._h), "jump_msd_mark")

    def msd(self, lj_only=False):
        """(1/N_sel) sum |x_i(now) - x_i(mark)|^2 on unwrapped positions, A^2."""
        out = C.c_double(0.0)
        self._check(self._L.jump_msd(self._h, int(bool(lj_only)), C.byref(out)), "jump_msd")
        return float(out.value)

    def vacf_mark(self):
        self._check(self._L.jump_vacf_mark(self._h), "jump_vacf_mark")

    def vacf_dot(self, lj_only=False):
        """(1/N_sel) sum v_i(mark) . v_i(now), (A/ps)^2."""
        c = C.c_double(0.0)
        self._check(self._L.jump_vacf_dot(self._h, int(bool(lj_only)), C.byref(c)), "jump_vacf_dot")
        return float(c.value)

    def slow_energy(self):
        e = C.c_double(0.0)
        self._check(self._L.jump_get_slow_energy(self._h, C.byref(e)), "jump_get_slow_energy")
        return float(e.value)

    def jump_half(self, H_ps, with_accel=True, step=0):
        self._check(self._L.jump_half(self._h, float(H_ps), int(bool(with_accel)), int(step)), "jump_half")

    def sync(self):
        self._check(self._L.jump_sync(self._h), "jump_sync")

    def refresh(self):
        self._check(self._L.jump_refresh(self._h), "jump_refresh")

    def refresh_lazy(self):
        """Re-read pos / vel; rows are rebuilt only if an atom left the skin/2 ball of its build position.  -> rebuilt?"""
        flag = C.c_int32(0)
        self._check(self._L.jump_refresh_lazy(self._h, C.byref(flag)), "jump_refresh_lazy")
        return bool(flag.value)

    def run_host(self, host_pos, host_vel, n_steps, mode="jump"):
        """End-to-end call with HOST state: copy (x, v) from the (pinned) host tensors to the device, take them over
        (jump_refresh_lazy: the rows are rebuilt at those positions unless every atom is still within skin/2 of where
        the last build saw it), run n_steps (mode "jump": jump_step; "respa": jump_respa_step with n_steps / n_inner
        outer steps; "baoab": baoab_step) and copy (x, v) back into the same host tensors.  The copies and kernels are
        enqueued on the context's stream (jump_refresh_lazy synchronises it once); the caller synchronises at the end."""
        torch = self._torch
        with torch.cuda.stream(self.stream):
            self.pos.copy_(host_pos, non_blocking=True)
            self.vel.copy_(host_vel, non_blocking=True)
            self.refresh_lazy()
            if mode == "jump":
                self.jump_step(n_steps)
            elif mode == "respa":
                self.jump_respa_step(max(int(n_steps) // int(self.params.n_inner), 1))
            elif mode == "baoab":
                self.baoab_step(n_steps)
            else:
                raise ValueError(mode)
            host_pos.copy_(self.pos, non_blocking=True)
            host_vel.copy_(self.vel, non_blocking=True)

    # ---- observers -----------------------------------------------------------------------------------
    def forces(self, which=0):
        out = self._torch.empty((self.n, 3), dtype=self._torch.float32, device=self.device)
        self._check(self._L.jump_get_forces(self._h, int(which), C.c_void_p(out.data_ptr())), "jump_get_forces")
        return out

    def energy(self):
        ek, ep = C.c_double(), C.c_double()
        self._check(self._L.jump_get_energy(self._h, C.byref(ek), C.byref(ep)), "jump_get_energy")
        return ek.value, ep.value

    def temperature(self):
        ek = C.c_double()
        self._check(self._L.jump_get_energy(self._h, C.byref(ek), None), "jump_get_energy")
        return 2.0 * ek.value / (3.0 * self.n * 1.987204259e-3)

    def stats(self):
        s = jump_stats()
        self._check(self._L.jump_get_stats(self._h, C.byref(s)), "jump_get_stats")
        d = {k: getattr(s, k) for k, _ in jump_stats._fields_ if k not in ("max_row", "cap_row", "pad")}
        d["max_row"], d["cap_row"] = list(s.max_row), list(s.cap_row)
        return d

    def reset_stats(self):
        self._check(self._L.jump_reset_stats(self._h), "jump_reset_stats")

    def events(self):
        n = C.c_int64()
        self._check(self._L.jump_get_events(self._h, None, 0, C.byref(n)), "jump_get_events")
        buf = np.zeros(int(n.value), dtype=EVENT_DTYPE)
        assert buf.itemsize == C.sizeof(jump_event)
        if n.value:
            self._check(self._L.jump_get_events(self._h, buf.ctypes.data_as(C.c_void_p), int(n.value), C.byref(n)), "jump_get_events")
        return np.sort(buf, order=["step", "stream", "atom", "iter"])

    def clear_events(self):
        self._check(self._L.jump_clear_events(self._h), "jump_clear_events")

    def row(self, which, atom):
        out = (C.c_int32 * self.n)()
        m = self._check(self._L.jump_get_row(self._h, int(which), int(atom), out, self.n), "jump_get_row")
        return np.frombuffer(out, dtype=np.int32, count=m).copy()

    def images(self):
        """Periodic image counters (n x 3 int32 on the device): unwrapped position = pos + images * box."""
        out = self._torch.empty((self.n, 3), dtype=self._torch.int32, device=self.device)
        self._check(self._L.jump_get_images(self._h, C.c_void_p(out.data_ptr())), "jump_get_images")
        return out

    def pos_unwrapped(self):
        box = self._torch.tensor([self.params.box[0], self.params.box[1], self.params.box[2]], dtype=self._torch.float64, device=self.device)
        return self.pos.double() + self.images().double() * box

    def rdf_accumulate(self, hist, r_max, lj_only=True):
        """Add the pair-distance histogram of the current positions to hist (device int64 / uint64 tensor of n_bins)."""
        assert hist.is_cuda and hist.element_size() == 8 and hist.is_contiguous()
        self._check(self._L.jump_rdf_accumulate(self._h, int(bool(lj_only)), float(r_max), int(hist.numel()),
                                                C.c_void_p(hist.data_ptr())), "jump_rdf_accumulate")

    def bounds(self):
        out = (C.c_double * 12)()
        self._check(self._L.jump_get_bounds(self._h, out), "jump_get_bounds")
        return dict(zip(["GM", "GL", "GV", "qmax", "eps_max", "sig_min", "sig_max", "rM", "G3", "GV2", "GV3", "rA"], list(out)))

    def set_lax_skin(self, on=True):
        """A displacement beyond skin/2 between two list builds is (not) an error."""
        self._check(self._L.jump_set_lax_skin(self._h, int(bool(on))), "jump_set_lax_skin")

    def set_lanes(self, lanes=0):
        """Lanes per jump chain in the update kernel (1, 4, 8, 16; 0 = automatic)."""
        self._check(self._L.jump_set_lanes(self._h, int(lanes)), "jump_set_lanes")

    def set_profiling(self, on=True):
        self._check(self._L.jump_set_profiling(self._h, int(bool(on))), "jump_set_profiling")

    def profile(self):
        """{category: (milliseconds, bracketed launches)} since profiling was switched on."""
        ms, cnt = (C.c_double * 4)(), (C.c_int64 * 4)()
        self._check(self._L.jump_get_profile(self._h, ms, cnt), "jump_get_profile")
        return {k: (ms[i], cnt[i]) for i, k in enumerate(("pair", "bonded", "update", "build"))}

    def count_pairs(self, which_row, r_cut):
        n = C.c_int64()
        self._check(self._L.jump_count_pairs(self._h, int(which_row), float(r_cut), C.byref(n)), "jump_count_pairs")
        return int(n.value)

    @property
    def step(self):
        return int(self._L.jump_get_step(self._h))

    @property
    def launches(self):
        return int(self._L.jump_get_launches(self._h))
