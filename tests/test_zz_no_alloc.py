"""jump_vacf_dot_static -- the velocity autocorrelation sum for callers that may not allocate (include/jump_b200.h):
scratch in a static device array of the library, no cudaMalloc.  Checked against the existing path
(jump_vacf_mark / jump_vacf_dot, which keeps its partial sums in a buffer of the context) on the same velocities, on
two calls in a row, to the relative tolerance the existing path's own test uses (1e-12: both are fp64 sums of the same
fp32 products, in a different order -- the context sums in cell-sorted order, this entry point in the caller's).

Collected last (test_zz_*): the suite runs with pytest -x, and a failure here must not hide another test.
"""
import numpy as np
import pytest

from paper_2412_15073_b200 import workloads as wl

pytestmark = pytest.mark.gpu
REL = 1e-12


@pytest.fixture(scope="module")
def jb():
    from paper_2412_15073_b200 import binding
    return binding


def test_static_scratch_entry_point_matches_the_context_path_twice(jb):
    import torch
    sysd, run = wl.make_config(0)
    g = jb.JumpSim(sysd, **run)
    g.vacf_mark()
    g.sync()
    v_origin = g.vel.clone()                                  # (n, 3) float32, original atom order
    oxy = torch.as_tensor((np.asarray(sysd["lj_eps"]) > 0).astype(np.int32), device=g.device)
    out = torch.full((2,), -1.0, dtype=torch.float64, device=g.device)
    n_sel = {None: g.n, "oxy": int(oxy.sum().item())}
    for call in range(2):                                     # two calls in a row share the static array
        g.jump_step(10 * (call + 1))                          # call 0: 10 steps; call 1: 20 more (across a re-sort)
        g.sync()
        want_all, want_oxy = g.vacf_dot(), g.vacf_dot(lj_only=True)
        v_now = g.vel.clone()
        jb.vacf_dot_static(v_now, v_origin, out)
        got = out.cpu().numpy().copy()
        assert got[1] == n_sel[None] and got[0] == pytest.approx(want_all, rel=REL), (call, got, want_all)
        jb.vacf_dot_static(v_now, v_origin, out, select=oxy)
        got = out.cpu().numpy().copy()
        assert got[1] == n_sel["oxy"] and got[0] == pytest.approx(want_oxy, rel=REL), (call, got, want_oxy)
        assert abs(want_all) > 1.0                            # (A/ps)^2: a real signal, not 0 == 0
    # a smaller problem right after a larger one: stale partial sums beyond ceil(n / 256) are never read
    m = 300
    jb.vacf_dot_static(v_now[:m].contiguous(), v_origin[:m].contiguous(), out)
    want = float((v_now[:m].double() * v_origin[:m].double()).sum().item()) / m
    got = out.cpu().numpy()
    assert got[1] == m and got[0] == pytest.approx(want, rel=1e-11)
    g.close()


def test_static_scratch_entry_point_rejects_sizes_beyond_its_array(jb):
    import torch
    n = jb.VACF_STATIC_MAX_ATOMS + 1
    v = torch.zeros((n, 3), dtype=torch.float32, device="cuda:0")
    out = torch.zeros(2, dtype=torch.float64, device="cuda:0")
    with pytest.raises(jb.JumpError, match="JUMP_VACF_STATIC_MAX_ATOMS"):
        jb.vacf_dot_static(v, v, out)
    # the limit itself is served: every atom with v = (1, 2, 2) gives 9 exactly
    v = torch.tensor([1.0, 2.0, 2.0], dtype=torch.float32, device="cuda:0").repeat(jb.VACF_STATIC_MAX_ATOMS, 1).contiguous()
    jb.vacf_dot_static(v, v, out)
    got = out.cpu().numpy()
    assert got[0] == 9.0 and got[1] == jb.VACF_STATIC_MAX_ATOMS
