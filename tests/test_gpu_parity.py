"""GPU parity: the CUDA path (through the C ABI of include/fargo.h) against the CPU oracle, element by
element, on the same seeded inputs.  Bar (BASELINE.json north_star):
    rel_f = max_active |gpu_f - oracle_f| / max_active |oracle_f|  <= 1e-10 (fp64), <= 1e-4 (fp32),
and the time step, which is a max/min reduction and therefore exact, must be BIT-equal.
Both sides keep automatic FMA contraction off and follow one operation order,
so in practice the fp64 fields come out bit-identical; the tests assert the contract's tolerance and
print the observed difference.
"""
import numpy as np
import pytest

import gpu_cases as G
from oracle.binding import Oracle
from paper_1602_02359_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL64 = 1e-10
TOL32 = 1e-4


def _gpu(w, precision=64, use_graph=True, kernel_plan=0):
    from paper_1602_02359_b200 import Fargo
    g = Fargo(w.mesh, w.geometry, w.eos, w.params, precision=precision, use_graph=use_graph, kernel_plan=kernel_plan)
    g.set_fields(*w.fields())
    return g


def _oracle(w):
    o = Oracle(w.mesh, w.geometry, w.eos, w.params)
    o.set_fields(*w.fields())
    return o


def _rel(a, b):
    d = float(np.max(np.abs(a.astype(np.float64) - b)))
    s = float(np.max(np.abs(b)))
    return d / s if s > 0 else d


def _diff_report(name, a, b):
    d = np.abs(a.astype(np.float64) - b)
    idx = np.unravel_index(int(np.argmax(d)), d.shape)
    return "%s: rel %.3e, max|d| %.3e at %s (gpu %.17g, oracle %.17g), %d / %d elements differ" % (
        name, _rel(a, b), float(d.max()), idx, float(a[idx]), float(b[idx]), int((d > 0).sum()), d.size)


# ---------------------------------------------------------------- per-stage parity (fp64) -------------
def _stage_arrays(w, stage):
    """(gpu name, oracle name) pairs holding defined data once `stage` has run."""
    adi = w.eos == W.ADIABATIC
    hx, hy, hz = w.mesh.nx > 1, w.mesh.ny > 1, w.mesh.nz > 1
    vel = [("vx", "vx")] + ([("vy", "vy")] if hy else []) + ([("vz", "vz")] if hz else [])
    mom = ([("pxm", "pxm"), ("pxp", "pxp")] if hx else []) + ([("pym", "pym"), ("pyp", "pyp")] if hy else []) + \
          ([("pzm", "pzm"), ("pzp", "pzp")] if hz else [])
    tr = [("trho", "rho")] + ([("te", "e")] if adi else []) + mom
    visc3 = w.params.nu > 0 and hx and hy and hz
    visc = visc3 or (w.params.nu > 0 and w.geometry == W.CYLINDRICAL and hx and hy and not hz)
    sfx = lambda s: ([("vx" + s, "vx" + s)] if hx else []) + ([("vy" + s, "vy" + s)] if hy else []) + \
        ([("vz" + s, "vz" + s)] if hz else [])
    return {
        "BC1": [("rho", "rho"), ("e", "e")] + vel,
        "VMEAN": [("v0", "v0")] if w.params.fargo_on else [],
        "POT": [("phi", "phi")] if (w.geometry != W.CARTESIAN and (w.params.gm_star or w.params.planet_mass)) else [],
        "DT": [],
        "SRC_A": sfx("b"),
        # adiabatic: 7b and 7c are one kernel (e_c is never stored): compared at the last stage it contains
        "SRC_B": [] if adi else sfx("c"),
        "SRC_C": (sfx("c") + [("ed", "ed")]) if adi else [],
        "SRC_D": ([("vxd", "vxd"), ("vyd", "vyd")] + ([("vzd", "vzd")] if visc3 else [])) if visc else [],
        "BC2": [("rho", "rho"), ("e", "e")] + vel,
        "SWEEP_X": tr if hx else [],
        "SWEEP_Y": tr if hy else [],
        "SWEEP_Z": tr if hz else [],
        "ORB_SHIFT": (tr + [("nshift", "nshift")]) if w.params.fargo_on else [],
    }[stage]


STAGES = ["BC1", "VMEAN", "POT", "DT", "SRC_A", "SRC_B", "SRC_C", "SRC_D", "BC2", "SWEEP_X", "SWEEP_Y", "SWEEP_Z",
          "ORB_SHIFT"]


@pytest.mark.parametrize("make", G.ALL, ids=[m.__name__ for m in G.ALL])
def test_stage_by_stage(make):
    """Every kernel alone: run both sides up to each stage of Fig. 2 and compare the arrays it wrote,
    ghost zones included (both sides compute wherever the stencil fits and pass the input through elsewhere)."""
    from paper_1602_02359_b200 import binding as B
    w = make()
    bad = []
    for stage in STAGES:
        pairs = _stage_arrays(w, stage)
        if not pairs and stage != "DT":
            continue
        # the kernel-per-cell sequence: it computes in the ghost zones too (the fused passes: test_fused_stages)
        o, g = _oracle(w), _gpu(w, use_graph=False, kernel_plan=B.PLAN_UNFUSED_SOURCE | B.PLAN_UNFUSED_VISC)
        o.step_until(stage)
        g.step_until(stage)
        if stage == "DT":
            dt_o, dt_g = o.time()[1], g.time()[1]
            if dt_o != dt_g:
                bad.append("DT: gpu %.17g oracle %.17g" % (dt_g, dt_o))
        for gn, on in pairs:
            a, b = g.array(gn), o.array(on)
            if _rel(a, b) > TOL64 or not np.isfinite(a).all():
                bad.append(stage + " " + _diff_report(gn, a, b))
        g.close(); o.close()
    assert not bad, "\n".join(bad)


@pytest.mark.parametrize("make", G.ALL, ids=[m.__name__ for m in G.ALL])
@pytest.mark.parametrize("use_graph", [False, True], ids=["stream", "graph"])
def test_multi_step(make, use_graph):
    """Several full updates (graph replay and plain launches): fields within 1e-10, clock bit-equal."""
    w = make()
    o, g = _oracle(w), _gpu(w, use_graph=use_graph)
    o.step(w.nsteps)
    g.step(w.nsteps)
    to, tg = o.time(), g.time()
    assert tg[2] == to[2]
    assert tg[0] == to[0] and tg[1] == to[1], "clock differs: gpu %r oracle %r" % (tg, to)
    fo, fg = o.get_fields(), g.get_fields()
    bad = []
    for name, a, b in zip(("rho", "e", "vx", "vy", "vz"), fg, fo):
        r = _rel(a, b)
        print("%s %s rel %.3e" % (w.name, name, r))
        if r > TOL64 or not np.isfinite(a).all():
            bad.append(_diff_report(name, a, b))
    assert not bad, "\n".join(bad)
    assert g.kernel_launches() > 0


FUSED_STAGES = [G.cart_adi_periodic_even, G.cart_iso_periodic, G.sph3d_iso_fargo, G.cyl3d_adi_fargo, G.sph3d_adi_nofargo,
                G.sheet3d_adi_fargo, G.cyl3d_visc_fargo, G.sph3d_visc_fargo, G.sheet3d_visc]


@pytest.mark.parametrize("make", FUSED_STAGES, ids=[m.__name__ for m in FUSED_STAGES])
def test_fused_stages(make):
    """The one-pass source step (k_source_fused) and the one-pass 7d (k_visc3d_fused) ALONE against the oracle:
    fargo_step_until takes them when fargo_step would, and they are observable at the last stage they contain
    (SRC_C: v_c and, adiabatic, e after 7c; SRC_D: v after 7d).  They produce active cells only (the ghost fill of cell
    9 follows), so the comparison is over the active cells."""
    w = make()
    visc = w.params.nu > 0
    adi = w.eos == W.ADIABATIC
    bad = []
    for stage, names in (("SRC_C", ["vxc", "vyc", "vzc"] + (["ed"] if adi else [])), ("SRC_D", ["vxd", "vyd", "vzd"] if visc else [])):
        if not names:
            continue
        o, g = _oracle(w), _gpu(w, use_graph=False)
        l0 = g.kernel_launches()
        o.step_until(stage)
        g.step_until(stage)
        # bc, [vmean], [potential], dt (2 kernels) + ONE source kernel (+ ONE 7d kernel): the unfused sequence has more
        unf = _gpu(w, use_graph=False, kernel_plan=3)
        u0 = unf.kernel_launches()
        unf.step_until(stage)
        assert g.kernel_launches() - l0 < unf.kernel_launches() - u0, "the fused pass did not run"
        unf.close()
        sl = tuple(slice(ng, ng + n) for ng, n in ((g.ngz, w.mesh.nz), (g.ngy, w.mesh.ny), (g.ngx, w.mesh.nx)))
        for nm in names:
            a, b = g.array(nm)[sl], o.array(nm)[sl]
            if _rel(a, b) > TOL64 or not np.isfinite(a).all():
                bad.append(stage + " " + _diff_report(nm, a, b))
        g.close(); o.close()
    assert not bad, "\n".join(bad)


FUSED = [G.cart_adi_periodic_even, G.cart_iso_periodic, G.sph3d_iso_fargo, G.cyl3d_adi_fargo, G.sph3d_adi_nofargo,
         G.sheet3d_adi_fargo]


@pytest.mark.parametrize("make", FUSED, ids=[m.__name__ for m in FUSED])
def test_fused_source_equals_the_kernel_sequence(make):
    """The one-pass source step (k_source_fused) against the 7a -> 7b -> 7c kernels it replaces (selected with
    fargo_params.kernel_plan = FARGO_PLAN_UNFUSED_SOURCE): bit-identical fields after several updates, and both within
    the bar of the oracle (test_multi_step)."""
    from paper_1602_02359_b200 import binding as B
    w = make()
    g1 = _gpu(w)
    g2 = _gpu(w, kernel_plan=B.PLAN_UNFUSED_SOURCE)
    g1.step(w.nsteps); g2.step(w.nsteps)
    assert g1.time() == g2.time()
    assert g1.kernel_launches() < g2.kernel_launches()      # the fused path really is the one that ran
    for name, a, b in zip(("rho", "e", "vx", "vy", "vz"), g1.get_fields(), g2.get_fields()):
        assert np.array_equal(a, b), _diff_report(name, a, b)


VISC_FUSED = [G.cyl3d_visc_fargo, G.sph3d_visc_fargo, G.sheet3d_visc]


@pytest.mark.parametrize("make", VISC_FUSED, ids=[m.__name__ for m in VISC_FUSED])
def test_fused_viscous_step_equals_the_kernel_sequence(make):
    """7a-7c in one pass (with the extra ghost layer) followed by 7d in one pass (k_visc3d_fused) against
    k_source_a -> k_source_b(c) -> k_visc3d_tensor -> k_visc3d_force (kernel_plan = FARGO_PLAN_UNFUSED_VISC):
    bit-identical fields."""
    from paper_1602_02359_b200 import binding as B
    w = make()
    g1 = _gpu(w)
    g1.step(w.nsteps)
    g2 = _gpu(w, kernel_plan=B.PLAN_UNFUSED_VISC)
    g2.step(w.nsteps)
    assert g1.time() == g2.time()
    assert g1.kernel_launches() < g2.kernel_launches()
    for name, a, b in zip(("rho", "e", "vx", "vy", "vz"), g1.get_fields(), g2.get_fields()):
        assert np.array_equal(a, b), _diff_report(name, a, b)


@pytest.mark.parametrize("make", [G.sheet3d_adi_fargo, G.sph3d_visc_fargo], ids=["sheet3d_adi_fargo", "sph3d_visc_fargo"])
def test_next1_cases_fp32(make):
    """fp32 build of the NEXT-1 paths (shearing sheet; fused 7d) against the fp64 oracle: <= 1e-4."""
    w = make()
    _run_config(w, w.nsteps, precision=32, tol=TOL32)


# ---------------------------------------------------------------- the five configs ---------------------
def _run_config(w, nsteps, precision=64, tol=TOL64):
    o, g = _oracle(w), _gpu(w, precision=precision)
    o.step(nsteps)
    g.step(nsteps)
    fo, fg = o.get_fields(), g.get_fields()
    rels = {}
    for name, a, b in zip(("rho", "e", "vx", "vy", "vz"), fg, fo):
        assert np.isfinite(a).all(), name
        rels[name] = _rel(a, b)
    print(w.name, "steps", o.time()[2], "t", o.time()[0], {k: "%.2e" % v for k, v in rels.items()})
    assert max(rels.values()) <= tol, rels
    return o, g


def test_config1_sound_wave():
    """Config 1: 32^3 linear sound wave, 200 steps; also the phase speed against the closed form."""
    w = W.sound_wave()
    o, g = _run_config(w, 200)
    assert g.time() == o.time()
    rho = g.get_fields()[0]
    m = w.mesh
    psi = 2 * np.pi * (m.xc()[None, None, :] + m.yc()[None, :, None] + m.zc()[:, None, None])
    a, b = np.sum((rho - 1) * np.cos(psi)), np.sum((rho - 1) * np.sin(psi))
    phase = np.arctan2(b, a) % (2 * np.pi)
    expect = (2 * np.pi * np.sqrt(3.0) * 1.0 * g.time()[0]) % (2 * np.pi)
    dphi = (phase - expect + np.pi) % (2 * np.pi) - np.pi
    assert abs(dphi) < 0.005 * 2 * np.pi * np.sqrt(3.0) * g.time()[0], (phase, expect)


def test_config2_sod():
    """Config 2: Sod tube 512x4x4 to t = 0.2 (outflow X = ghosted X axis)."""
    w = W.sod()
    o, g = _run_config(w, 2000)
    assert g.time() == o.time() and g.time()[0] == 0.2


def test_config3_disk2d():
    """Config 3: 768x256 cylindrical isothermal disk, planet, viscosity, FARGO; 500 steps."""
    w = W.disk2d()
    _run_config(w, 500)


def test_config4_disk3d_reduced():
    """Config 4 at a size the oracle finishes in seconds (192x64x16, same recipe); the full size is
    checked by test_full_size.py on sampled rings."""
    w = W.disk3d(192, 64, 16)
    _run_config(w, 30)


def test_config5_noise_box_64():
    w = W.noise_box(64)
    _run_config(w, 50)


def test_config5_noise_box_64_fp32():
    """fp32 build against the fp64 oracle: <= 1e-4."""
    w = W.noise_box(64)
    _run_config(w, 50, precision=32, tol=TOL32)


# ---------------------------------------------------------------- edge cases -----------------------------
def test_uniform_state_is_preserved():
    w = W.noise_box(shape3=(40, 8, 8))
    w.rho[...] = 1.0; w.vx[...] = 0.25; w.vy[...] = -0.5; w.vz[...] = 0.125
    g = _gpu(w)
    g.step(5)
    rho, e, vx, vy, vz = g.get_fields()
    assert np.all(rho == 1.0) and np.all(e == w.e) and np.all(vx == 0.25) and np.all(vy == -0.5) and np.all(vz == 0.125)


@pytest.mark.parametrize("make", [G.cyl2d_iso_fargo_visc, G.sph3d_iso_fargo, G.cyl3d_adi_fargo],
                         ids=["cyl2d_iso_fargo_visc", "sph3d_iso_fargo", "cyl3d_adi_fargo"])
def test_second_set_fields_keeps_the_static_potential(make):
    """Restart path: fargo_set_fields clears the arrays (the stored potential among them); on a context whose graph
    already exists the potential must be written again before the next replay.  set, step, set, step == a fresh
    context == the oracle."""
    w = make()
    g = _gpu(w)
    g.step(2)
    g.set_fields(*w.fields())
    g.step(w.nsteps)
    o = _oracle(w)
    o.step(w.nsteps)
    assert g.time() == o.time()
    for name, a, b in zip(("rho", "e", "vx", "vy", "vz"), g.get_fields(), o.get_fields()):
        assert _rel(a, b) <= TOL64, _diff_report(name, a, b)


def test_set_get_roundtrip_and_device_pointers():
    """fargo_get_fields(fargo_set_fields(x)) == x bit for bit (the checkpoint path), host and device pointers."""
    import torch
    w = G.cart_adi_mixed_bc()
    g = _gpu(w)
    for a, b in zip(g.get_fields(), w.fields()):
        assert np.array_equal(a, b)
    dev = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in w.fields()]
    g.set_fields(*dev)
    out = [torch.empty_like(t) for t in dev]
    g.get_fields(out)
    for a, b in zip(out, dev):
        assert torch.equal(a, b)


def test_t_stop_makes_later_steps_noops():
    w = G.sod_small()
    o, g = _oracle(w), _gpu(w)
    o.step(60); g.step(60)
    assert g.time() == o.time() and g.time()[0] == 0.05
    f1 = g.get_fields()
    g.step(3)
    for a, b in zip(g.get_fields(), f1):
        assert np.array_equal(a, b)


def test_exact_integer_shift():
    """delta v = 0 and v0 dt / LX an exact integer: the ring is rotated bit for bit."""
    import math
    nphi, nr = 64, 8
    bc = ((W.PERIODIC,) * 2, (W.REFLECTING,) * 2, (W.PERIODIC,) * 2)
    mesh = W.Mesh(nphi, nr, 1, 0.0, 2.0 * math.pi, W.uedges(1.0, 2.0, nr), np.array([-0.5, 0.5]), bc)
    prm = W.Params(fargo_on=1, dt_fixed=0.25)
    shape = (1, nr, nphi)
    r = mesh.yc()[None, :, None] * np.ones(shape)
    rho = 1.0 + 0.3 * W.uniform_pm1(0, nr * nphi).reshape(shape)
    cs = np.full(shape, 1e-3)
    nsh = np.array([3, -2, 5, 0, 1, -7, 64, 2])[None, :, None]
    vx = nsh * (mesh.dx * r) / prm.dt_fixed * np.ones(shape)
    w = W.Workload("shift", mesh, W.CYLINDRICAL, W.ISOTHERMAL, prm, rho, cs, vx, np.zeros(shape), None, 1)
    g, o = _gpu(w, use_graph=False), _oracle(w)
    g.step_until("ORB_SHIFT"); o.step_until("ORB_SHIFT")
    got, ref = g.array("trho"), o.array("rho")
    assert np.array_equal(g.array("nshift"), o.array("nshift"))
    assert np.array_equal(got, ref)


def test_division_is_correctly_rounded():
    """The kernels' branch-free division (csrc/common.cuh rdiv) against IEEE division on the host: bit-equal on
    2^24 random operand pairs spanning 2^+-400 in each operand plus a set of hard cases."""
    import torch
    from paper_1602_02359_b200.binding import selftest_div
    rng = np.random.default_rng(20260211)
    n = 1 << 24
    def draw():
        m = rng.uniform(1.0, 2.0, n)
        e = rng.integers(-400, 400, n)
        s = rng.choice([-1.0, 1.0], n)
        return s * np.ldexp(m, e)
    a, b = draw(), draw()
    # hard cases: quotients next to rounding boundaries, equal operands, powers of two, zero numerators
    k = np.arange(1, 4097, dtype=np.float64)
    a[:4096] = k; b[:4096] = 3.0
    a[4096:8192] = 1.0; b[4096:8192] = 1.0 + k * 2.0 ** -52
    a[8192:12288] = 1.0 + k * 2.0 ** -52; b[8192:12288] = 1.0 + (k + 1) * 2.0 ** -52
    a[12288:16384] = 0.0
    a[16384:20480] = b[16384:20480]
    b[20480:24576] = 6.0
    got = selftest_div(torch.from_numpy(a).cuda(), torch.from_numpy(b).cuda()).cpu().numpy()
    ref = a / b
    bad = np.nonzero(got != ref)[0]
    assert bad.size == 0, "first mismatch: %r / %r -> gpu %r host %r (%d of %d)" % (
        a[bad[0]], b[bad[0]], got[bad[0]], ref[bad[0]], bad.size, n)
    # the division by the constant six of the PPA step (rdiv6): same operands, plus multiples of 6 +- 1 ulp
    a[:4096] = 6.0 * k; a[4096:8192] = np.nextafter(6.0 * k, np.inf); a[8192:12288] = np.nextafter(6.0 * k, -np.inf)
    got6 = selftest_div(torch.from_numpy(a).cuda()).cpu().numpy()
    ref6 = a / 6.0
    bad = np.nonzero(got6 != ref6)[0]
    assert bad.size == 0, "rdiv6 first mismatch: %r / 6 -> gpu %r host %r (%d of %d)" % (
        a[bad[0]], got6[bad[0]], ref6[bad[0]], bad.size, n)


GUARDED = [G.cart_adi_periodic_even, G.sph3d_iso_fargo, G.cart_adi_mixed_bc, G.cyl3d_visc_fargo, G.sheet3d_adi_fargo, G.sod_small,
           G.yz_only_2d, G.sph3d_iso_fargo_odd]


@pytest.mark.parametrize("make", GUARDED, ids=[m.__name__ for m in GUARDED])
def test_nothing_is_written_outside_the_workspace(make):
    """compute-sanitizer is closed on this GPU pool (profiles/r02b_final.md), so out-of-bounds writes are looked for with
    1 MiB canary regions before and after the workspace: several updates through every kernel family (fused and
    kernel-per-cell plans, both precisions), field I/O and the inspection calls must leave them untouched."""
    from paper_1602_02359_b200 import Fargo
    w = make()
    for precision in (64, 32):
        for plan in (0, 7):
            g = Fargo(w.mesh, w.geometry, w.eos, w.params, precision=precision, kernel_plan=plan, guard_bytes=1 << 20)
            g.set_fields(*w.fields())
            g.step(3)
            g.get_fields()
            g.diagnostics()
            g.step_until("SWEEP_X")
            g.array("trho")
            assert g.check_guards(), (w.name, precision, plan)
            g.close()
