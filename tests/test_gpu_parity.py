"""GPU-vs-oracle parity through the C ABI (libppm_b200.so) — `pytest -m gpu` on a B200.

Bars (BASELINE.json north_star; norms in tests/parity_norms.py):
  max relative error per variable <= 1e-5 after one step, <= 1e-4 after the config's step count on smooth
  flows; L1 error <= 1e-4 on the shock config; conserved totals within 1e-6 relative; dt within 1e-6.
Every input comes from the seeded generators in paper_1810_13416_b200.workloads; no expected value comes
from the CUDA path.  Full-size configs (128^3 .. 1024^3) are checked on oracle WINDOWS: the update reaches 4
cells per axis per step, so a window plus a 4*steps apron regenerated from the input formulas reproduces the
global result on the window exactly (tests/test_oracle_invariants.py::test_window_reproduces_full_grid).
"""
import numpy as np
import pytest
import torch

from paper_1810_13416_b200 import workloads as W

from parity_norms import conserved_rel, l1_rel, max_rel, merge_scales, pert_rel

pytestmark = pytest.mark.gpu

ONE_STEP, MULTI_STEP, L1_SHOCK, CONS, DT_TOL = 1e-5, 1e-4, 1e-4, 1e-6, 1e-6
# The perturbation fields rho' = rho - rho0, p' = p - p0 compared directly (ppm_get_state in perturbation form against the
# oracle's stored perturbations), relative to max |rho'|, max |p'|: the bar for the low-Mach gravity configs, where the
# full-value norm above would let rho', p' be wrong by their own size.  fp32 carries 6e-8 of the FULL rho, p
# through every flux difference, i.e. 6e-8 / (max|q'| / q0) of the perturbation per operation; DESIGN.md section 2 (R20b).
PERT_TOL = 1e-4       # measured on a B200: <= 5.1e-6 on every config (profiles/r2_parity_perturbation.md)


def _gpu():
    from paper_1810_13416_b200.binding import PPM       # loads libppm_b200.so; raises if missing
    return PPM


def _oracle(w, n=None, org=(0, 0, 0), bc=None):
    from oracle import binding as ob
    n = n or (w.n, w.n, w.n)
    return ob.Oracle(n[0], n[1], n[2], w.dx, w.gamma, bc or w.bc, w.grav, org=org, rho_floor=w.rho_floor, p_floor=w.p_floor)


def _load(g, w, device="cuda", nzs=32):
    n = w.n
    for z0 in range(0, n, nzs):
        z1 = min(n, z0 + nzs)
        g.set_state(w.fields((0, 0, z0), (n, n, z1), device=device), z0=z0)


def _run_pair(w, steps, chunk=0, check_each=(), flat3d=False, direct=False, twofluid=None, edit=None):
    """steps on both sides with the GPU's dt; returns dict of results after step 1 and at the end.
    twofluid = (gamma_tracked, gamma_rest): NEXT-4 on both sides; edit(f): in-place change of the input fields."""
    PPM = _gpu()
    from paper_1810_13416_b200.binding import OPT_FLATTEN3D, OPT_IO_PATH
    f = w.fields()
    if edit is not None:
        edit(f)
    o = _oracle(w)
    if twofluid:
        o.set_two_fluid(*twofluid)
    o.set_state(f.numpy())
    g = PPM.from_workload(w)
    if chunk:
        g.set_chunk(chunk)
    if flat3d:                      # SURVEY 8(f) NEXT-1 on both sides
        g.set_option(OPT_FLATTEN3D, 1)
        o.set_flatten3d(True)
    if direct:
        g.set_option(OPT_IO_PATH, 1)
    if twofluid:
        g.set_two_fluid(*twofluid)
    g.set_state(f.cuda())
    out = {}
    c0g, c0o = g.reduce_conserved(), o.reduce_conserved()
    full0 = o.get_state()
    out["cons0"] = conserved_rel(c0g, c0o, full0, w.dx, w.gamma)
    for s in range(steps):
        dt = g.cfl_dt(w.cfl)
        assert abs(dt - o.cfl_dt(w.cfl)) <= DT_TOL * dt
        order = 0 if s % 2 == 0 else 5
        g.step(dt, order)
        o.step(dt, order)
        if s == 0 or s + 1 == steps or (s + 1) in check_each:
            gs = g.get_state().cpu().numpy().astype(np.float64)
            os_ = o.get_state()
            out[s + 1] = (max_rel(gs, os_), l1_rel(gs, os_))
    out["cons1"] = conserved_rel(g.reduce_conserved(), o.reduce_conserved(), o.get_state(), w.dx, w.gamma)
    # the perturbation fields as stored on both sides (no base state added, no rounding of rho0 + rho')
    from paper_1810_13416_b200.binding import OPT_STATE_FORM
    g.set_option(OPT_STATE_FORM, 1)
    gp = g.get_state().cpu().numpy().astype(np.float64)
    g.set_option(OPT_STATE_FORM, 0)
    out["pert"] = pert_rel((gp[0], gp[4]), (o.raw_field(0), o.raw_field(4)))
    print("perturbation-form parity after %d steps (%s %d^3): %s" % (steps, w.name, w.n, {k: float("%.3g" % v) for k, v in out["pert"].items()}))
    fmt = lambda e: {k: float("%.2e" % v) for k, v in e.items()}
    print("parity %s %d^3%s: max-rel after 1 step %s; after %d steps max-rel %s, L1 %s; conserved totals %.1e" % (
        w.name, w.n, " (two-fluid)" if twofluid else (" (3-D flattening)" if flat3d else ""), fmt(out[1][0]), steps, fmt(out[steps][0]),
        fmt(out[steps][1]), float(out["cons1"].max())))
    # R20a keeps one scale (max |m000|) for the ten FV coefficients; the margin against each coefficient's OWN maximum stays
    # visible here (a coefficient that vanishes by symmetry has no scale of its own and reports 0)
    own = [float(np.abs(gs[5 + k] - os_[5 + k]).max() / np.abs(os_[5 + k]).max()) if np.abs(os_[5 + k]).max() > 1e-6 * np.abs(os_[5]).max() else 0.0
           for k in range(10)]
    print("   FV coefficients against their own maxima (m000 m100 m010 m001 m200 m020 m002 m110 m101 m011): %s" % " ".join("%.1e" % v for v in own))
    out["drift_gpu"] = np.abs(g.reduce_conserved() - c0g)
    out["c0"] = c0g
    out["final"] = (gs, os_)
    g.close()
    return out


# ---------------------------------------------------------------- config 1: the full config -----------
def test_cfg1_full_32cubed_20_steps():
    w = W.make(1)
    r = _run_pair(w, w.steps)
    assert max(r[1][0].values()) <= ONE_STEP, r[1][0]
    assert max(r[w.steps][0].values()) <= MULTI_STEP, r[w.steps][0]
    assert r["cons0"].max() <= CONS and r["cons1"].max() <= CONS
    # the scheme is conservative on the periodic box: mass, energy, tracked mass drift only by fp32 round-off
    c0, d = r["c0"], r["drift_gpu"]
    assert d[0] <= 2e-6 * c0[0] and d[4] <= 2e-6 * c0[4] and d[5] <= 2e-6 * c0[5]
    fv = r["final"][0][5]
    assert fv.min() >= 0.0 and fv.max() <= 1.0


def test_data_paths_agree():
    """the bulk-staged sweeps (default when the extent along the sweep axis is whole bricks) and the direct
    global-memory sweeps run the same marching body on the same brick records: bit-identical results."""
    PPM = _gpu()
    from paper_1810_13416_b200.binding import OPT_IO_PATH
    for cfg, n in ((1, 32), (4, 32), (3, 32), (2, 32), (1, 40)):     # 40: 10 brick columns, the last warp of a CTA row is half empty
        w = W.make(cfg, n=n)
        f = w.fields().cuda()
        res = []
        for mode in ("bulk", "direct"):
            g = PPM.from_workload(w)
            if mode == "direct":
                g.set_option(OPT_IO_PATH, 1)
            assert [g.axis_path(d) for d in range(3)] == [1 if mode == "bulk" else 0] * 3
            g.set_state(f)
            for s in range(3):
                g.step(g.cfl_dt(0.8), s * 2)
            res.append(g.get_state().cpu().numpy().astype(np.float64))
            g.close()
        assert np.array_equal(res[0], res[1])


@pytest.mark.parametrize("chunk", [8, 13])
def test_pencil_chunking_does_not_change_results(chunk):
    PPM = _gpu()
    w = W.make(1)
    f = w.fields().cuda()
    res = []
    for ch in (0, chunk):
        g = PPM.from_workload(w)
        g.set_chunk(ch)
        g.set_state(f)
        for s in range(2):
            g.step(0.02, s * 5)
        res.append(g.get_state().cpu().numpy())
        g.close()
    assert np.array_equal(res[0], res[1])


def test_cfl_reduction_fused_into_the_last_sweep_equals_the_standalone_pass():
    """the last sweep of ppm_step reduces max_d |u_d| + c of the state it writes, so ppm_cfl_dt launches
    nothing after a step.  The standalone pass (PPM_OPT_CFL_FUSED = 0, and always after ppm_set_state / ppm_sweep) uses the
    same formula on the stored state: without a base state the two maxima are the same bits; with one, the sweep's full
    pressure comes from its (rho, p) window instead of a fresh table lookup and they agree to fp32 rounding."""
    PPM = _gpu()
    from paper_1810_13416_b200.binding import OPT_CFL_FUSED
    for cfg, n, tol in ((1, 32, 0.0), (3, 32, 0.0), (4, 32, 3e-7), (2, 32, 3e-7)):
        w = W.make(cfg, n=n)
        f = w.fields().cuda()
        dts = {}
        for fused in (1, 0):
            g = PPM.from_workload(w)
            g.set_option(OPT_CFL_FUSED, fused)
            g.set_state(f)
            dts[fused] = []
            n0 = g.launch_count()
            for s in range(4):
                dt = g.cfl_dt(w.cfl)
                dts[fused].append(dt)
                g.step(dts[1][s], s)                      # both runs take the same steps
            dts[fused].append(g.cfl_dt(w.cfl))
            # launches: fused = 1 pass after set_state + 4 x 3 sweeps; standalone = 5 passes + 12 sweeps
            assert g.launch_count() - n0 == (13 if fused else 17)
            state = g.get_state().cpu().numpy()
            g.close()
            dts[(fused, "state")] = state
        assert np.array_equal(dts[(1, "state")], dts[(0, "state")])
        a, b = np.array(dts[1]), np.array(dts[0])
        assert a[0] == b[0]                                # both from the standalone pass after set_state
        if tol == 0.0:
            assert np.array_equal(a, b), (cfg, a, b)
        else:
            assert np.max(np.abs(a - b) / b) <= tol, (cfg, a, b)
        assert len(set(a)) == len(a)                       # the maximum really changes from step to step


def test_uniform_fv_shortcut_gives_the_same_values():
    """PPM_OPT_FV_SHORTCUT: where FV is uniform under a whole warp the PPB remap is skipped; the values must be those of the
    full remap (bit for bit, up to the sign of a zero), on a state where the shortcut fires in most places (config 4: FV = 0 / 1
    away from r = 0.45), on one where it fires almost nowhere (config 1) and on a constructed one with exactly uniform slabs."""
    PPM = _gpu()
    from paper_1810_13416_b200.binding import OPT_FV_SHORTCUT
    for cfg, n, steps, tf in ((4, 64, 8, None), (1, 32, 6, None), (4, 64, 6, TWO_FLUID)):
        w = W.make(cfg, n=n)
        f = w.fields()
        if cfg == 4:
            f[5:, :, :, :20] = 0.0                      # an exactly uniform slab next to the varying field
            f[5, :, :, :20] = 0.25
        res = []
        for on in (1, 0):
            g = PPM.from_workload(w)
            if tf:
                g.set_two_fluid(*tf)                    # (the two-fluid sweeps take the shortcut too)
            g.set_option(OPT_FV_SHORTCUT, on)
            g.set_state(f.cuda())
            for s in range(steps):
                g.step(g.cfl_dt(w.cfl), s % 6)
            res.append(g.get_state())
            g.close()
        assert torch.equal(res[0], res[1]), float((res[0] - res[1]).abs().max())
        assert float(res[0][6:].abs().max()) > 0.0


# ---------------------------------------------------------------- reduced-size, full step counts ------
def test_cfg2_stratified_reduced_64_100_steps():
    w = W.make(2, n=64)
    r = _run_pair(w, 100)
    assert max(r[1][0].values()) <= ONE_STEP, r[1][0]
    assert max(r[100][0].values()) <= MULTI_STEP, r[100][0]
    assert r["cons1"].max() <= CONS
    assert r["pert"]["rho'"] <= PERT_TOL and r["pert"]["p'"] <= PERT_TOL, r["pert"]


def test_cfg3_blast_reduced_64_50_steps_L1():
    w = W.make(3, n=64)
    r = _run_pair(w, 50)
    assert max(r[1][1].values()) <= L1_SHOCK, r[1][1]
    assert max(r[50][1].values()) <= L1_SHOCK, r[50][1]
    assert r["cons1"].max() <= CONS
    gs, os_ = r["final"]
    assert np.abs(os_[1:4]).max() > 3.0           # the Mach ~3 blast really ran
    assert gs[5].min() >= 0.0 and gs[5].max() <= 1.0


# ---------------------------------------------------------------- NEXT-1: fully 3-D shock flattening --
@pytest.mark.parametrize("direct", [False, True])
def test_flatten3d_blast_matches_oracle(direct):
    """config 3 (Mach ~3 blast through a 1000:1 density jump) in the 3-D flattening mode, both data
    paths: the detector kernel + the sweeps that read its field against the oracle's 3-D mode."""
    w = W.make(3, n=48)
    r = _run_pair(w, 40, flat3d=True, direct=direct)
    assert max(r[1][1].values()) <= L1_SHOCK, r[1][1]
    assert max(r[40][1].values()) <= L1_SHOCK, r[40][1]
    assert r["cons1"].max() <= CONS
    # the mode really differs from the 1-D one on this flow (else the test would prove nothing)
    r1 = _run_pair(w, 40)
    d = l1_rel(r["final"][0], r1["final"][0])
    assert max(d.values()) > 20 * L1_SHOCK, d


def test_flatten3d_smooth_flow_equals_1d_mode_bitwise():
    """no shock anywhere (config 1): F~ = 0 and the 3-D mode must reproduce the 1-D mode bit for bit"""
    PPM = _gpu()
    from paper_1810_13416_b200.binding import OPT_FLATTEN3D
    w = W.make(1)
    f = w.fields().cuda()
    res = []
    for mode in (0, 1):
        g = PPM.from_workload(w)
        g.set_option(OPT_FLATTEN3D, mode)
        g.set_state(f)
        for s in range(3):
            g.step(g.cfl_dt(0.8), s * 2)
        res.append(g.get_state().cpu().numpy())
        assert g.launch_count() == (3 * (3 + mode) + 1 + 2)       # per step: 3 sweeps (+ 1 detector); 1 cfl pass (the others are fused into the sweeps); set + get
        g.close()
    assert np.array_equal(res[0], res[1])


def test_flatten3d_ragged_grid_and_paths_agree():
    PPM = _gpu()
    from oracle import binding as ob
    from paper_1810_13416_b200.binding import OPT_FLATTEN3D, OPT_IO_PATH
    rng = np.random.default_rng(12)
    nx, ny, nz = 36, 30, 22
    f = np.zeros((15, nz, ny, nx), dtype=np.float32)
    f[0] = 1.0 + rng.random((nz, ny, nx))
    f[1:4] = 0.25 * rng.normal(size=(3, nz, ny, nx))
    f[4] = np.exp(0.6 * rng.normal(size=(nz, ny, nx)))        # pressure jumps: the detector is on in many cells
    f[5] = 0.2 + 0.6 * rng.random((nz, ny, nx))
    bc = (1, 1, 0, 0, 1, 1)
    o = ob.Oracle(nx, ny, nz, 0.03, 1.4, bc, None)
    o.set_flatten3d(True)
    o.set_state(f)
    assert (o.flatten3d_field() > 0.5).mean() > 0.02
    res = []
    for io in (0, 1):
        g = PPM(nx, ny, nz, 0.03, 1.4, bc)
        g.set_option(OPT_FLATTEN3D, 1)
        g.set_option(OPT_IO_PATH, io)
        g.set_state(f)
        dts = []
        for order in (0, 3, 5):
            dt = 0.4 * g.cfl_dt(0.8)
            dts.append(dt)
            g.step(dt, order)
        res.append(g.get_state().cpu().numpy().astype(np.float64))
        g.close()
    assert np.array_equal(res[0], res[1])
    for dt, order in zip(dts, (0, 3, 5)):
        o.step(dt, order)
    e = l1_rel(res[0], o.get_state())
    assert max(e.values()) <= L1_SHOCK, e


# ---------------------------------------------------------------- NEXT-2: PPB-only advection ----------
def test_advect_matches_oracle_and_paths_agree():
    """PPB-only steps (ppm_advect) on config 1's fields (32^3 periodic) and on a ragged grid with mirror walls: FV
    against the oracle's mode, the hydro fields bit for bit untouched, bulk-staged == direct bitwise."""
    PPM = _gpu()
    from oracle import binding as ob
    from paper_1810_13416_b200.binding import OPT_IO_PATH
    rng = np.random.default_rng(31)
    cases = []
    w = W.make(1)
    f1 = w.fields().numpy()
    f1[1:4] *= 8.0                                             # Courant numbers up to ~0.5 at dt below
    cases.append((f1, (w.n,) * 3, w.dx, w.bc, 0.5 * w.dx / np.abs(f1[1:4]).max()))
    nx, ny, nz = 36, 30, 22
    f2 = np.zeros((15, nz, ny, nx), dtype=np.float32)
    f2[0], f2[4] = 1.0, 1.0
    f2[1:4] = 0.5 * rng.normal(size=(3, nz, ny, nx))
    f2[5] = 0.2 + 0.6 * rng.random((nz, ny, nx))
    f2[6:] = 0.02 * rng.normal(size=(9, nz, ny, nx))
    cases.append((f2, (nx, ny, nz), 0.03, (1, 1, 0, 0, 1, 1), 0.4 * 0.03 / np.abs(f2[1:4]).max()))
    for f, dims, dx, bc, dt in cases:
        o = ob.Oracle(dims[0], dims[1], dims[2], dx, 1.4, bc, None)
        o.set_state(f)
        for order in range(6):
            o.advect(dt, order)
        os_ = o.get_state()
        res = []
        for io in (0, 1):
            g = PPM(dims[0], dims[1], dims[2], dx, 1.4, bc)
            g.set_option(OPT_IO_PATH, io)
            g.set_state(f)
            h0 = g.get_state().cpu().numpy()
            n0 = g.launch_count()
            for order in range(6):
                g.advect(dt, order)
            assert g.launch_count() - n0 == 18
            res.append(g.get_state().cpu().numpy())
            assert np.array_equal(res[-1][:5], h0[:5])          # the hydro state is held fixed
            g.close()
        assert np.array_equal(res[0], res[1])
        e = max_rel(res[0].astype(np.float64), os_)
        assert e["FV"] <= ONE_STEP, e
        assert np.abs(os_[5] - f[5]).max() > 1e-3               # ... and FV really moved


def test_advect_split_state_mixes_with_every_other_call():
    """the bulk-staged PPB-only sweeps write the PPB part of the brick records only, so after an odd number of them the hydro
    fields and the PPB coefficients sit in different buffers until something else looks at the state (ppm_make_whole):
    interleaved with full steps, single sweeps, partial loads, reductions and reads, the bulk-staged path must return bit
    for bit what the direct path (whole records in every sweep) returns"""
    PPM = _gpu()
    from paper_1810_13416_b200.binding import OPT_IO_PATH
    w = W.make(1)
    f = w.fields().numpy()
    f[1:4] *= 4.0
    dt = 0.3 * w.dx / (np.abs(f[1:4]).max() + np.sqrt(1.4 * f[4].max() / f[0].min()))
    res = []
    for io in (0, 1):
        g = PPM.from_workload(w)
        g.set_option(OPT_IO_PATH, io)
        g.set_state(f)
        out = []
        g.advect(dt, 0)                                   # 3 sweeps: split
        out.append(g.get_state().cpu().numpy())           # read of a split state
        assert np.array_equal(out[-1][:5], f[:5])
        g.advect(dt, 1)
        g.step(dt, 2)                                     # full step on a split state
        g.advect(dt, 3)
        out.append(np.array([g.cfl_dt(0.8)]))             # reduction over a split state
        g.advect(dt, 4)
        g.advect(dt, 5)                                   # even number: whole again without a copy
        g.sweep(dt, 1)
        g.advect(dt, 0)
        out.append(g.reduce_conserved())
        g.advect(dt, 2)
        g.set_state(np.ascontiguousarray(f[:, 8:16]), z0=8)     # partial load (z-planes 8..15) into a split state
        g.advect(dt, 1)
        out.append(g.get_state().cpu().numpy())
        res.append(out)
        g.close()
    for a, b in zip(res[0], res[1]):
        assert np.array_equal(a, b)
    assert not np.array_equal(res[0][0][5], f[5])


def test_advect_slotted_disc_one_revolution_fig3():
    """PAPER.md Fig. 3 on the paper's grid: 100 x 100 cells (x 1: the 2-D case, six in-plane coefficients), one
    revolution = 1256 PPB-only steps, against the oracle.  The field is a 0/1 indicator, so the bar is the L1 one."""
    PPM = _gpu()
    from oracle import binding as ob
    n, steps = 100, 1256
    f = W.slotted_disc(n)
    dt = 1.0 / steps
    o = ob.Oracle(n, n, 1, 1.0 / n, 1.4, (0,) * 6)
    g = PPM(n, n, 1, 1.0 / n, 1.4, (0,) * 6)
    o.set_state(f)
    g.set_state(f)
    for k in range(steps):
        order = 0 if k % 2 == 0 else 2
        o.advect(dt, order)
        g.advect(dt, order)
    gs = g.get_state().cpu().numpy().astype(np.float64)
    os_ = o.get_state()
    g.close()
    e = l1_rel(gs, os_)
    assert e["FV"] <= L1_SHOCK, e
    assert gs[5].min() >= 0.0 and gs[5].max() <= 1.0
    assert abs(gs[5].sum() - f[5].astype(np.float64).sum()) <= 1e-5 * f[5].sum()      # fp32 round-off of 2512 sweeps
    # the disc is back: slot still open, bridge still full (the oracle pins carry the comparison with donor-cell)
    assert gs[5, 0, 64:78, 49:51].max() < 0.12 and gs[5, 0, 64:78, 43:45].min() > 0.9
    assert not gs[[8, 11, 13, 14]].any()                       # the out-of-plane coefficients stay zero: the 6-moment 2-D scheme


def test_advect_slotted_disc_holds_for_100_revolutions_fig3():
    """PAPER.md Fig. 3 shows the disc at 0, 1, 10 and 100 revolutions and L43 says the scheme holds it.  One revolution is
    checked against the oracle above; the oracle would need ten minutes for a hundred, so this is a property test of
    the GPU path on the paper's own sequence (125,600 PPB-only steps, 377k launches, a few seconds): the slot stays
    open, the solid parts stay full, FV stays in [0,1], its integral is conserved to fp32 round-off, and after 100
    revolutions the error is still several times below what first-order advection has after ONE (0.066, pinned in
    tests/test_oracle_advect.py)."""
    PPM = _gpu()
    n, steps = 100, 1256
    f = W.slotted_disc(n)
    m0 = f[5, 0].astype(np.float64)
    dt = 1.0 / steps
    g = PPM(n, n, 1, 1.0 / n, 1.4, (0,) * 6)
    g.set_state(f)
    done, l1 = 0, {}
    for target, slot_max, solid_min in ((1, 0.12, 0.93), (10, 0.15, 0.92), (100, 0.30, 0.88)):
        for k in range((target - done) * steps):
            g.advect(dt, 0 if k % 2 == 0 else 2)
        done = target
        s = g.get_state().cpu().numpy().astype(np.float64)
        fv = s[5, 0]
        l1[target] = np.abs(fv - m0).sum() / m0.size
        assert fv.min() >= 0.0 and fv.max() <= 1.0
        assert abs(fv.sum() - m0.sum()) <= 1e-6 * m0.sum()
        assert fv[64:78, 49:51].max() < slot_max, (target, fv[64:78, 49:51].max())
        assert min(fv[64:78, 43:45].min(), fv[64:78, 55:57].min()) > solid_min, target
        assert not s[[8, 11, 13, 14]].any()
    g.close()
    assert l1[1] < 0.012 and l1[10] < 0.015 and l1[100] < 0.02, l1          # measured 0.0103, 0.0124, 0.0174


def test_cfg4_convection_reduced_64_20_steps():
    w = W.make(4, n=64)
    r = _run_pair(w, 20)
    assert max(r[1][0].values()) <= ONE_STEP, r[1][0]
    assert max(r[20][0].values()) <= MULTI_STEP, r[20][0]
    assert r["cons1"].max() <= CONS
    assert r["pert"]["rho'"] <= PERT_TOL and r["pert"]["p'"] <= PERT_TOL, r["pert"]


@pytest.mark.parametrize("dims", [(37, 29, 23), (36, 30, 22)])
def test_ragged_grid_all_boundaries_and_orders(dims):
    """extents that are not multiples of the 4-cell brick (pad cells in the last bricks, half-empty warps), mixed
    boundaries, all six orders.  (36, 30, 22): nx % 4 == 0, so the x sweep takes the bulk-staged path over ragged y, z."""
    PPM = _gpu()
    from oracle import binding as ob
    rng = np.random.default_rng(11)
    nx, ny, nz = dims
    f = np.zeros((15, nz, ny, nx), dtype=np.float32)
    f[0] = 1.0 + 0.3 * rng.random((nz, ny, nx))
    f[1:4] = 0.2 * rng.normal(size=(3, nz, ny, nx))
    f[4] = 0.8 + 0.3 * rng.random((nz, ny, nx))
    f[5] = 0.2 + 0.6 * rng.random((nz, ny, nx))
    f[6:] = 0.02 * rng.normal(size=(9, nz, ny, nx))
    P_, R_ = 0, 1
    for bc in ((P_, P_, R_, R_, P_, P_), (R_, R_, P_, P_, R_, R_)):
        o = ob.Oracle(nx, ny, nz, 0.03, 1.4, bc, None)
        g = PPM(nx, ny, nz, 0.03, 1.4, bc)
        assert [g.axis_path(d) for d in range(3)] == [int(e % 4 == 0) for e in (nx, ny, nz)]
        o.set_state(f)
        g.set_state(f)
        for order in range(6):
            dt = 0.4 * g.cfl_dt(0.8)
            g.step(dt, order)
            o.step(dt, order)
        e = max_rel(g.get_state().cpu().numpy().astype(np.float64), o.get_state())
        assert max(e.values()) <= MULTI_STEP, e
        g.close()


@pytest.mark.parametrize("dims", [(16, 8, 1), (12, 1, 1), (1, 1, 9), (5, 3, 2), (8, 4, 4)])
def test_degenerate_grids_2d_1d_and_fewer_cells_than_ghosts(dims):
    """quasi-2-D and 1-D grids (one brick thick, mostly pad cells) and periodic axes with fewer cells than the 4
    ghost cells a sweep reaches (the images wrap around more than once)."""
    PPM = _gpu()
    from oracle import binding as ob
    rng = np.random.default_rng(21)
    nx, ny, nz = dims
    f = np.zeros((15, nz, ny, nx), dtype=np.float32)
    f[0] = 1.0 + 0.3 * rng.random((nz, ny, nx))
    f[1:4] = 0.2 * rng.normal(size=(3, nz, ny, nx))
    f[4] = 0.8 + 0.3 * rng.random((nz, ny, nx))
    f[5] = 0.2 + 0.6 * rng.random((nz, ny, nx))
    f[6:] = 0.02 * rng.normal(size=(9, nz, ny, nx))
    bc = (0,) * 6
    o = ob.Oracle(nx, ny, nz, 0.05, 1.4, bc, None)
    g = PPM(nx, ny, nz, 0.05, 1.4, bc)
    o.set_state(f)
    g.set_state(f)
    for order in (0, 5, 2):
        dt = 0.5 * g.cfl_dt(0.8)
        g.step(dt, order)
        o.step(dt, order)
    e = max_rel(g.get_state().cpu().numpy().astype(np.float64), o.get_state())
    assert max(e.values()) <= MULTI_STEP, e
    c = g.reduce_conserved()
    assert np.all(np.isfinite(c))
    g.close()


def _synthetic_gravity(kind, dims, dx, rng):
    """a smooth, mildly stratified base state with its table (hand-made, not hydrostatically exact: the scheme must
    agree with the oracle for ANY table; the residual just acts as a source)"""
    nx, ny, nz = dims
    if kind == 1:                                   # CONST_Z: nodes on every cell centre and face, ghosts included
        n = 2 * (nz + 8) + 1
        s0, ds = -4 * dx, 0.5 * dx
        z = s0 + ds * np.arange(n)
        center = (0.0, 0.0, 0.0)
    else:                                           # RADIAL about an off-centre point
        n = 257
        s0, ds = 0.0, 2.0 * dx * max(dims) / (n - 1)
        z = s0 + ds * np.arange(n)
        center = (0.45 * nx * dx, 0.55 * ny * dx, 0.5 * nz * dx)
    H = 2.0 * dx * max(dims)
    rho0 = (1.0 + 0.5 * np.exp(-z / H)).astype(np.float32)
    p0 = (0.8 + 0.4 * np.exp(-z / H)).astype(np.float32)
    g = (-0.3 * np.exp(-z / H) * (np.tanh(z / (2 * dx)) if kind == 2 else 1.0)).astype(np.float32)
    return dict(kind=kind, s0=float(s0), ds=float(ds), center=center, g=g, rho0=rho0, p0=p0)


@pytest.mark.parametrize("seed", range(8))
def test_random_small_grids_boundaries_gravity_and_paths(seed):
    """randomised: extents 1..21 per axis (whole-brick and ragged axes mixed, so bulk-staged and direct sweeps mix in
    one step), every boundary combination, no / constant-z / radial gravity tables, both flattening modes, random sweep
    orders — against the oracle, and bulk-staged == direct bitwise."""
    PPM = _gpu()
    from oracle import binding as ob
    from paper_1810_13416_b200.binding import OPT_FLATTEN3D, OPT_IO_PATH
    rng = np.random.default_rng(1000 + seed)
    pool = [1, 2, 3, 4, 5, 7, 8, 9, 12, 13, 16, 20, 21]
    dims = tuple(int(rng.choice(pool)) for _ in range(3))
    bc = []
    for d in range(3):
        refl = bool(rng.integers(0, 2)) and dims[d] >= 4
        bc += [1, 1] if refl else [0, 0]
    kind = int(rng.integers(0, 3))
    dx = 0.05
    grav = _synthetic_gravity(kind, dims, dx, rng) if kind else None
    flat = int(rng.integers(0, 2))
    nx, ny, nz = dims
    f = np.zeros((15, nz, ny, nx), dtype=np.float32)
    f[0] = 1.6 + 0.3 * rng.random((nz, ny, nx))
    f[1:4] = 0.2 * rng.normal(size=(3, nz, ny, nx))
    f[4] = 1.3 + 0.3 * rng.random((nz, ny, nx))
    f[5] = 0.2 + 0.6 * rng.random((nz, ny, nx))
    f[6:] = 0.02 * rng.normal(size=(9, nz, ny, nx))
    orders = [int(rng.integers(0, 6)) for _ in range(3)]
    o = ob.Oracle(nx, ny, nz, dx, 1.4, bc, grav)
    o.set_flatten3d(bool(flat))
    o.set_state(f)
    res, dts = [], []
    for io in (0, 1):
        g = PPM(nx, ny, nz, dx, 1.4, bc, grav)
        g.set_option(OPT_IO_PATH, io)
        g.set_option(OPT_FLATTEN3D, flat)
        g.set_state(f)
        for k, order in enumerate(orders):
            if io == 0:
                dts.append(0.5 * g.cfl_dt(0.8))
            g.step(dts[k], order)
        res.append(g.get_state().cpu().numpy().astype(np.float64))
        g.close()
    assert np.array_equal(res[0], res[1]), (dims, bc, kind, flat)
    for dt, order in zip(dts, orders):
        o.step(dt, order)
    e = max_rel(res[0], o.get_state())
    assert max(e.values()) <= MULTI_STEP, (dims, bc, kind, flat, e)


def test_state_flag_reports_floor_hits_and_bad_states():
    """error behaviour of the boundary (include/ppm.h): a step that drives the pressure to its floor, or a state with
    non-positive density, is reported as PPM_ESTATE by the next synchronising call; a new ppm_set_state clears it."""
    PPM = _gpu()
    from paper_1810_13416_b200.binding import PPMError, PPM_ESTATE
    n = 16
    f = np.zeros((15, n, n, n), dtype=np.float32)
    f[0], f[4], f[5] = 1.0, 1.0, 0.5
    g = PPM(n, n, n, 1.0 / n, 1.4, (0,) * 6, p_floor=1e-6, rho_floor=1e-6)
    g.set_state(f)
    g.step(0.5 * g.cfl_dt(0.8), 0)
    g.sync()                                               # a healthy state: no flag
    bad = f.copy()
    bad[1, :, :, : n // 2] = 30.0                          # Mach 25 streams pulling apart: a near-vacuum opens between them
    bad[1, :, :, n // 2:] = -30.0
    bad[1] *= -1.0
    g.set_state(bad)
    dt = g.cfl_dt(0.8)
    for s in range(6):
        g.step(4.0 * dt, 0)                                # and a time step far beyond the CFL limit
    with pytest.raises(PPMError) as ei:
        g.sync()
    assert ei.value.code == PPM_ESTATE
    g.set_state(f)                                         # loading a state clears the sticky flag
    g.sync()
    neg = f.copy()
    neg[0, 3, 4, 5] = -1.0
    g.set_state(neg)
    with pytest.raises(PPMError) as ei:
        g.cfl_dt(0.8)
    assert ei.value.code == PPM_ESTATE
    g.close()


def test_host_pipelined_exchange_equals_serial_set_step_get():
    """the end-to-end helper of bench.py's e2e leg (binding.PPM.step_host_pipelined: slab-wise upload of grid s+1 on one copy
    stream while grid s comes down on another, ppm_set_state / ppm_get_state with device staging slabs) returns bit for
    bit what ppm_set_state(host) -> ppm_step -> ppm_get_state(host) returns, ragged last slab included"""
    PPM = _gpu()
    w = W.make(4, n=40)
    f0 = w.fields()
    f1 = f0.clone()
    f1[1:4] *= 0.5
    ins = [f0.pin_memory(), f1.pin_memory(), f0.pin_memory()]
    g = PPM.from_workload(w)
    g.set_state(f0.cuda())
    dt = 0.7 * g.cfl_dt(w.cfl)
    ref = []
    for s, fi in enumerate(ins):
        g.set_state(fi)
        g.step(dt, s)
        ref.append(g.get_state(device="cpu").numpy().copy())
    outs = [torch.empty_like(fi).pin_memory() for fi in ins]
    g.step_host_pipelined(ins, outs, dt, [0, 1, 2], slab=16)
    for r, o in zip(ref, outs):
        assert np.array_equal(r, o.numpy())
    assert not np.array_equal(ref[0], ref[1])
    # two contexts on two streams, every other grid each, nothing waited for until both are enqueued (bench.py's e2e leg)
    g2 = PPM.from_workload(w, stream=torch.cuda.Stream())
    outs2 = [torch.zeros_like(fi).pin_memory() for fi in ins]
    g.step_host_pipelined(ins[0::2], outs2[0::2], dt, [0, 2], slab=16, wait=False)
    g2.step_host_pipelined(ins[1::2], outs2[1::2], dt, [1], slab=16, wait=False)
    g.finish_host_pipelined()
    g2.finish_host_pipelined()
    for r, o in zip(ref, outs2):
        assert np.array_equal(r, o.numpy())
    g2.close()
    g.close()


def test_hydrostatic_state_is_preserved_exactly_on_gpu():
    PPM = _gpu()
    for cfg, n in ((2, 32), (4, 32)):
        w = W.make(cfg, n=n)
        f = w.fields()
        f[1:4] = 0.0
        g = PPM.from_workload(w)
        g.set_state(f.cuda())
        s0 = g.get_state().cpu().numpy()
        for s in range(3):
            g.step(0.8 * w.dx, s)
        s1 = g.get_state().cpu().numpy()
        if cfg == 2:      # rho', p' are exactly 0: bit-for-bit well-balanced
            assert np.array_equal(s0[:5], s1[:5])
        else:             # rho', p' = fp32 rounding of the input (~3e-8): only that noise evolves
            assert np.abs(s1[1:4]).max() < 2e-7 and np.abs(s1[0] - s0[0]).max() < 3e-7
        g.close()


# ---------------------------------------------------------------- NEXT-3: confining sphere, spin-up ---
def test_sphere_random_flow_matches_oracle_and_solid_cells_are_untouched():
    """violent random flow inside an off-centre sphere (reading R23): fluid cells against the oracle's sphere
    mode, solid cells bit for bit what was loaded, mass of the fluid conserved, all six sweep orders"""
    PPM = _gpu()
    from oracle import binding as ob
    rng = np.random.default_rng(41)
    n = 24
    f = np.zeros((15, n, n, n), dtype=np.float32)
    f[0] = 1.0 + 0.3 * rng.random((n, n, n))
    f[1:4] = 0.3 * rng.normal(size=(3, n, n, n))
    f[4] = 0.8 + 0.3 * rng.random((n, n, n))
    f[5] = 0.2 + 0.6 * rng.random((n, n, n))
    f[6:] = 0.02 * rng.normal(size=(9, n, n, n))
    for rad, cen in ((0.47, (0.5, 0.52, 0.48)), (0.5, (0.5, 0.5, 0.5)), (0.12, (0.3, 0.6, 0.5))):     # the last: segments of 1..6 cells
        o = ob.Oracle(n, n, n, 1.0 / n, 1.4, (1,) * 6, None)
        g = PPM(n, n, n, 1.0 / n, 1.4, (1,) * 6)
        o.set_sphere(rad, cen)
        g.set_sphere(rad, cen)
        o.set_state(f)
        g.set_state(f)
        m = o.solid_mask()
        c0 = g.reduce_conserved()
        assert abs(c0[0] - o.reduce_conserved()[0]) <= 1e-6 * c0[0]
        for order in range(6):
            dt = 0.5 * g.cfl_dt(0.8)
            assert abs(dt - 0.5 * o.cfl_dt(0.8)) <= DT_TOL * dt
            g.step(dt, order)
            o.step(dt, order)
        gs = g.get_state().cpu().numpy()
        os_ = o.get_state()
        assert np.array_equal(gs[:, m], f[:, m])
        fl = ~m
        e = max_rel(gs[:, fl].astype(np.float64)[:, None, None, :], os_[:, fl][:, None, None, :])
        assert max(e.values()) <= MULTI_STEP, (rad, e)
        c1 = g.reduce_conserved()
        assert abs(c1[0] - c0[0]) <= 3e-6 * c0[0] and abs(c1[5] - c0[5]) <= 3e-6 * c0[5]
        g.close()


def test_sphere_cfg4_star_in_its_sphere_64_20_steps():
    """config 4 in the paper's run geometry: the star inside the sphere inscribed in the cube, gravity
    already tapered to zero before it; 64^3, the config's 20 steps, with the spin-up ramp running during the first ten"""
    PPM = _gpu()
    w = W.make(4, n=64)
    f = w.fields()
    o = _oracle(w)
    g = PPM.from_workload(w)
    o.set_sphere(0.5, (0.5, 0.5, 0.5))
    g.set_sphere(0.5, (0.5, 0.5, 0.5))
    o.set_state(f.numpy())
    g.set_state(f.cuda())
    m = o.solid_mask()
    for s in range(20):
        if s < 10:
            g.spin_up(0.02)
            o.spin_up(0.02)
        dt = g.cfl_dt(w.cfl)
        assert abs(dt - o.cfl_dt(w.cfl)) <= DT_TOL * dt
        g.step(dt, 0 if s % 2 == 0 else 5)
        o.step(dt, 0 if s % 2 == 0 else 5)
        if s == 0:
            e1 = max_rel(g.get_state().cpu().numpy().astype(np.float64)[:, ~m][:, None, None, :], o.get_state()[:, ~m][:, None, None, :])
            assert max(e1.values()) <= ONE_STEP, e1
    gs = g.get_state().cpu().numpy()
    os_ = o.get_state()
    assert np.array_equal(gs[:, m], f.numpy()[:, m])
    e = max_rel(gs[:, ~m].astype(np.float64)[:, None, None, :], os_[:, ~m][:, None, None, :])
    assert max(e.values()) <= MULTI_STEP, e
    assert conserved_rel(g.reduce_conserved(), o.reduce_conserved(), np.where(m, 0.0, os_), w.dx, w.gamma).max() <= CONS
    x = (np.arange(64) + 0.5) / 64 - 0.5
    assert np.abs(os_[2][32, 32, :] - 0.2 * x).max() < 0.1 and np.abs(os_[2][32, 32, 40]) > 0.01        # it rotates
    g.close()


def test_sphere_cfg4_full_512_windows_that_straddle_the_sphere():
    """the headline grid in the sphere geometry, bench launch configuration: windows at a pole of the sphere, on its 45-degree
    flank, and in the shell, two steps, oracle windows with the same sphere"""
    c = 256
    _window_check(4, 2, [((c + 248, c, c), 24), ((c + 178, c + 178, c), 24), ((c + 150, c + 140, c + 150), 24), ((c + 175, c, c), 24)],
                  sphere=(0.5, (0.5, 0.5, 0.5)))


# ---------------------------------------------------------------- NEXT-4: two-fluid equation of state ------
TWO_FLUID = (1.4, 5.0 / 3.0)        # tracked fluid (FV), the rest


@pytest.mark.parametrize("direct", [False, True])
def test_two_fluid_cfg1_matches_oracle(direct):
    """config 1 (periodic, FV = tanh slab between 0.1 and 0.9: every cell is a mixture, Gamma varies between 1.43 and 1.63)
    with the velocities raised to Mach 0.3 so that the energy equation really works; 20 steps, both data paths"""
    w = W.make(1)

    def edit(f):
        f[1:4] *= 8.0
    r = _run_pair(w, w.steps, twofluid=TWO_FLUID, direct=direct, edit=edit)
    assert max(r[1][0].values()) <= ONE_STEP, r[1][0]
    assert max(r[w.steps][0].values()) <= MULTI_STEP, r[w.steps][0]
    assert r["cons0"].max() <= CONS and r["cons1"].max() <= CONS
    # the mixture's total energy sum(p beta(f) + KE) is conserved on the periodic box (fp32 round-off only)
    c0, d = r["c0"], r["drift_gpu"]
    assert d[0] <= 2e-6 * c0[0] and d[4] <= 2e-6 * c0[4] and d[5] <= 2e-6 * c0[5]
    print("two-fluid cfg1 (%s path): after 1 step %s, after %d steps %s" % ("direct" if direct else "bulk", r[1][0], w.steps, r[w.steps][0]))


def test_two_fluid_differs_from_single_fluid_and_equal_gammas_do_not():
    """the mode really changes the flow (so the test above is not vacuous), and with gamma_tracked = gamma_rest it is the
    single-fluid scheme to fp32 round-off"""
    PPM = _gpu()
    w = W.make(1)
    f = w.fields()
    f[1:4] *= 8.0
    res = []
    for tf in (None, (w.gamma, w.gamma), TWO_FLUID):
        g = PPM.from_workload(w)
        if tf:
            g.set_two_fluid(*tf)
        g.set_state(f.cuda())
        for s in range(5):
            g.step(0.004, s)
        res.append(g.get_state().cpu().numpy().astype(np.float64))
        g.close()
    e_same = max_rel(res[1], res[0])
    e_diff = max_rel(res[2], res[0])
    assert max(e_same.values()) <= 2e-6, e_same
    assert e_diff["p"] > 1e-3, e_diff


def test_two_fluid_blast_through_a_gas_interface_L1():
    """config 3 at 64^3 (Mach-3 blast, density contrast 1000) with the dense layer made of the OTHER gas (FV = the interface
    tanh instead of 1e-5 of it): shocks, the limiter and the Newton iterations with one Gamma per side; 30 steps"""
    w = W.make(3, n=64)

    def edit(f):
        f[5:] *= 1e5
    r = _run_pair(w, 30, twofluid=TWO_FLUID, edit=edit)
    assert max(r[1][1].values()) <= L1_SHOCK, r[1][1]
    assert max(r[30][1].values()) <= L1_SHOCK, r[30][1]
    assert r["cons1"].max() <= CONS
    gs, os_ = r["final"]
    assert np.abs(os_[1:4]).max() > 2.0 and os_[5].max() > 0.99
    print("two-fluid blast: L1 after 1 step %s, after 30 steps %s" % (r[1][1], r[30][1]))


def test_two_fluid_stratified_box_with_gravity():
    """config 2 at 64^3 (constant gravity, reflecting z walls, FV = 1 above z = 0.6): the hydrostatic base state does not depend
    on the gases' adiabatic indices, the perturbation equations do; 40 steps"""
    w = W.make(2, n=64)
    r = _run_pair(w, 40, twofluid=TWO_FLUID)
    assert max(r[1][0].values()) <= ONE_STEP, r[1][0]
    assert max(r[40][0].values()) <= MULTI_STEP, r[40][0]
    assert r["cons1"].max() <= CONS
    assert r["pert"]["rho'"] <= PERT_TOL and r["pert"]["p'"] <= PERT_TOL, r["pert"]


def test_two_fluid_radial_gravity_convection_zone():
    """config 4 at 64^3 (radial gravity, FV = 1 outside r = 0.45): the stable layer is the other gas; 10 steps"""
    w = W.make(4, n=64)
    r = _run_pair(w, 10, twofluid=TWO_FLUID)
    assert max(r[1][0].values()) <= ONE_STEP, r[1][0]
    assert max(r[10][0].values()) <= MULTI_STEP, r[10][0]
    assert r["cons1"].max() <= CONS
    assert r["pert"]["rho'"] <= PERT_TOL and r["pert"]["p'"] <= PERT_TOL, r["pert"]


def test_two_fluid_ragged_grid_mixed_boundaries():
    """37 x 29 x 24: direct path along x and y (ragged), bulk along z; reflecting x, periodic y, reflecting z"""
    PPM = _gpu()
    from oracle import binding as ob
    rng = np.random.default_rng(77)
    nx, ny, nz = 37, 29, 24
    dx = 1.0 / 40
    bc = (1, 1, 0, 0, 1, 1)
    f = torch.zeros((15, nz, ny, nx), dtype=torch.float32)
    z, y, x = np.meshgrid((np.arange(nz) + 0.5) * dx, (np.arange(ny) + 0.5) * dx, (np.arange(nx) + 0.5) * dx, indexing="ij")
    f[0] = torch.from_numpy(1.0 + 0.3 * np.sin(7 * x) * np.cos(5 * y) + 0.2 * np.sin(9 * z))
    f[4] = torch.from_numpy(0.8 + 0.2 * np.cos(6 * x + 4 * z))
    for k in (1, 2, 3):
        f[k] = torch.from_numpy(0.3 * np.sin(5 * x + 3 * y + 4 * z + k))
    f[5] = torch.from_numpy(0.5 + 0.45 * np.tanh((np.sin(6 * x) + np.cos(5 * y) + np.sin(4 * z)) / 0.3))
    f[6:] = torch.from_numpy(0.01 * rng.standard_normal((9, nz, ny, nx)))
    g = PPM(nx, ny, nz, dx, 5.0 / 3.0, bc)
    g.set_two_fluid(*TWO_FLUID)
    g.set_state(f.cuda())
    o = ob.Oracle(nx, ny, nz, dx, 5.0 / 3.0, bc, None)
    o.set_two_fluid(*TWO_FLUID)
    o.set_state(f.numpy())
    for s in range(6):
        dt = g.cfl_dt(0.6)
        assert abs(dt - o.cfl_dt(0.6)) <= DT_TOL * dt
        g.step(dt, s)
        o.step(dt, s)
        if s == 0:
            e1 = max_rel(g.get_state().cpu().numpy().astype(np.float64), o.get_state())
            assert max(e1.values()) <= ONE_STEP, e1
    e = max_rel(g.get_state().cpu().numpy().astype(np.float64), o.get_state())
    assert max(e.values()) <= MULTI_STEP, e
    assert conserved_rel(g.reduce_conserved(), o.reduce_conserved(), o.get_state(), dx, 5.0 / 3.0).max() <= CONS
    g.close()


def test_two_fluid_cfl_dt_sees_fv_moved_by_ppb_only_sweeps():
    """with two gases the sound speed depends on FV: after PPB-only sweeps ppm_cfl_dt must not return the maximum cached
    by the last full step (a one-cell spike of the stiffer gas spreads out, so the fastest signal slows down)"""
    PPM = _gpu()
    n = 16
    f = np.zeros((15, n, n, n), dtype=np.float32)
    f[0], f[4] = 1.0, 1.0
    f[1] = 0.3                                            # uniform translation along x
    f[5, 8, 8, 8] = 1.0
    g = PPM(n, n, n, 1.0 / n, 1.2, (0,) * 6)
    g.set_two_fluid(3.0, 1.2)
    g.set_state(f)
    dt = 0.2 * g.cfl_dt(0.8)
    g.step(dt, 0)                                         # leaves the maximum of its final state on the device
    dt_a = g.cfl_dt(0.8)
    for k in range(6):
        g.advect(dt, k % 6)
    dt_b = g.cfl_dt(0.8)
    st = g.get_state()
    h = PPM(n, n, n, 1.0 / n, 1.2, (0,) * 6)
    h.set_two_fluid(3.0, 1.2)
    h.set_state(st)
    assert dt_b == h.cfl_dt(0.8)
    assert dt_b > dt_a * 1.0001
    g.close()
    h.close()


def test_two_fluid_argument_checks():
    PPM = _gpu()
    from paper_1810_13416_b200.binding import OPT_FLATTEN3D
    w = W.make(4, n=32)
    g = PPM.from_workload(w)
    with pytest.raises(Exception):
        g.set_two_fluid(0.9, 1.4)                       # an adiabatic index <= 1
    g.set_two_fluid(*TWO_FLUID)
    with pytest.raises(Exception):
        g.set_sphere(0.5, (0.5, 0.5, 0.5))              # the two NEXT modes are not combined
    with pytest.raises(Exception):
        g.set_option(OPT_FLATTEN3D, 1)
    g.set_two_fluid(0.0)                                # off again
    g.set_sphere(0.5, (0.5, 0.5, 0.5))
    with pytest.raises(Exception):
        g.set_two_fluid(*TWO_FLUID)
    g.close()


# ---------------------------------------------------------------- NEXT-4: brick decomposition -------------
@pytest.mark.parametrize("cfg,n,procs,steps", [(4, 64, (2, 2, 2), 6), (1, 32, (2, 1, 2), 6), (2, 64, (2, 2, 1), 6), (4, 64, (1, 4, 1), 3)])
def test_brick_decomposition_equals_the_undivided_grid_bitwise(cfg, n, procs, steps):
    """the grid cut into sub-domains with PPM_BC_HALO faces, one brick layer exchanged
    with the two face neighbours before every sweep (all sub-domains in this process on this GPU, device copies for the
    messages) gives the SAME BITS as the undivided grid: radial gravity with walls (2x2x2 = the 8-GPU layout, and 4 slabs),
    the periodic cube (wrap-around neighbours, both neighbours the same sub-domain), plane-parallel gravity cut across x, y"""
    PPM = _gpu()
    from paper_1810_13416_b200.decomposition import BrickDecomposition, LocalCluster
    w = W.make(cfg, n=n)
    f = w.fields()
    mono = PPM.from_workload(w)
    mono.set_state(f.cuda())
    d = BrickDecomposition((n, n, n), procs, w.bc)
    cl = LocalCluster(d, w.dx, w.gamma, w.grav, w.rho_floor, w.p_floor)
    cl.set_state(f)
    assert torch.equal(cl.get_state(), mono.get_state())
    for s in range(steps):
        dt = mono.cfl_dt(w.cfl)
        assert cl.cfl_dt(w.cfl) == dt                       # the fused / standalone maxima of the parts bracket the same cells
        order = (0, 5, 2, 3)[s % 4]
        mono.step(dt, order)
        cl.step(dt, order)
    a, b = mono.get_state(), cl.get_state()
    assert torch.equal(a, b), float((a - b).abs().max())
    ca, cb = mono.reduce_conserved(), cl.reduce_conserved()
    assert np.allclose(ca, cb, rtol=1e-12, atol=1e-14 * np.abs(ca).max())
    # what travelled: per step, every cut axis sends 2 layers per interior face pair; nothing else
    sent = sum(p.halo_bytes for p in cl.parts)
    faces = sum(1 for r in range(d.size) for ax in range(3) for sd in (0, 1) if d.neighbour(r, ax, sd) is not None and True)
    per_step = sum(d.halo_cells(ax) * 15 * 4 for r in range(d.size) for ax in range(3) for sd in (0, 1) if d.neighbour(r, ax, sd) is not None)
    assert sent == steps * per_step and faces > 0
    mono.close()
    cl.close()


def test_brick_decomposition_argument_checks():
    PPM = _gpu()
    from paper_1810_13416_b200.binding import BC_HALO, OPT_FLATTEN3D, PPMError
    g = PPM(32, 32, 32, 1.0 / 32, 5.0 / 3.0, (1, BC_HALO, 1, 1, 1, 1))
    g.set_state(torch.ones((15, 32, 32, 32), dtype=torch.float32).cuda())
    with pytest.raises(PPMError):
        g.step(1e-3, 0)                                     # an exchange is due between the sweeps
    with pytest.raises(PPMError):
        g.sweep(1e-3, 0)                                    # no halo layer handed over yet
    g.sweep(1e-3, 1)                                        # axes without a HALO face sweep as ever
    lay = torch.empty(g.halo_floats(0), dtype=torch.float32, device="cuda")
    assert g.halo_floats(0) == 15 * 64 * 8 * 8
    with pytest.raises(PPMError):
        g.set_halo(0, 0, lay)                               # that face is a wall
    g.pack_halo(0, 0, lay)
    g.set_halo(0, 1, lay)
    g.sweep(1e-3, 0)
    g.sync()
    with pytest.raises(PPMError):
        PPM(30, 32, 32, 1.0 / 32, 5.0 / 3.0, (1, BC_HALO, 1, 1, 1, 1))      # not whole bricks along a HALO axis
    g.close()


# ---------------------------------------------------------------- full-size configs on windows --------
def _window_check(cfg, steps, windows, nzs_load=16, tol=ONE_STEP, norm="max", sphere=None):
    PPM = _gpu()
    w = W.make(cfg)
    n = w.n
    g = PPM.from_workload(w)
    if sphere:
        g.set_sphere(*sphere)
    _load(g, w, nzs=nzs_load)
    dts = []
    for s in range(steps):
        dt = g.cfl_dt(w.cfl)
        dts.append(dt)
        g.step(dt, 0 if s % 2 == 0 else 5)
    g.sync()
    apron = 4 * steps
    worst = {}
    pairs, perts = [], []
    for (c, size) in windows:
        lo = [max(0, c[d] - size // 2 - apron) for d in range(3)]
        hi = [min(n, c[d] + size // 2 + apron) for d in range(3)]
        bc = []
        for d in range(3):
            bc += [w.bc[2 * d] if lo[d] == 0 and (w.bc[2 * d] == 1 or hi[d] == n) else 2,
                   w.bc[2 * d + 1] if hi[d] == n and (w.bc[2 * d + 1] == 1 or lo[d] == 0) else 2]
        o = _oracle(w, n=[hi[d] - lo[d] for d in range(3)], org=lo, bc=bc)
        if sphere:
            o.set_sphere(*sphere)
        o.set_state(w.fields(lo, hi, device="cuda").cpu().numpy())
        for s, dt in enumerate(dts):
            o.step(dt, 0 if s % 2 == 0 else 5)
        os_ = o.get_state()
        # interior of the window: drop the apron on OPEN sides only
        sl = [slice(apron if bc[2 * d] == 2 else 0, (hi[d] - lo[d]) - (apron if bc[2 * d + 1] == 2 else 0)) for d in range(3)]
        zs = slice(lo[2] + sl[2].start, lo[2] + sl[2].stop)
        gs = g.get_state(z0=zs.start, nzs=zs.stop - zs.start).cpu().numpy().astype(np.float64)
        gs = gs[:, :, lo[1] + sl[1].start:lo[1] + sl[1].stop, lo[0] + sl[0].start:lo[0] + sl[0].stop]
        os_ = os_[:, sl[2], sl[1], sl[0]]
        pairs.append((gs, os_))
        if w.grav is not None and norm == "max":
            # the perturbation fields as both sides store them (PERT_TOL above)
            from paper_1810_13416_b200.binding import OPT_STATE_FORM
            g.set_option(OPT_STATE_FORM, 1)
            gp = g.get_state(z0=zs.start, nzs=zs.stop - zs.start).cpu().numpy().astype(np.float64)
            g.set_option(OPT_STATE_FORM, 0)
            gp = gp[:, :, lo[1] + sl[1].start:lo[1] + sl[1].stop, lo[0] + sl[0].start:lo[0] + sl[0].stop]
            perts.append(((gp[0], gp[4]), (o.raw_field(0)[sl[2], sl[1], sl[0]].copy(), o.raw_field(4)[sl[2], sl[1], sl[0]].copy())))
    g.close()
    scale = merge_scales([o_ for _, o_ in pairs])      # a window in a quiescent region has no scale of its own
    for gs, os_ in pairs:
        e = max_rel(gs, os_, scale) if norm == "max" else l1_rel(gs, os_)
        for k, v in e.items():
            worst[k] = max(worst.get(k, 0.0), v)
    print("parity cfg %d at full size (%d^3), %d windows, %d steps, %s norm: %s" % (cfg, n, len(windows), steps, norm, {k: float("%.2e" % v) for k, v in worst.items()}))
    assert max(worst.values()) <= tol, worst
    if perts:
        # scale = the largest perturbation over all windows (a window in the quiescent core has none of its own)
        sc = [max(np.abs(op[k]).max() for _, op in perts) for k in (0, 1)]
        pe = [max(np.abs(gp[k] - op[k]).max() for gp, op in perts) / sc[k] if sc[k] > 0 else 0.0 for k in (0, 1)]
        print("perturbation-form parity, cfg %d windows after %d steps: rho' %.3g (scale %.3g), p' %.3g (scale %.3g)" % (cfg, steps, pe[0], sc[0], pe[1], sc[1]))
        assert max(pe) <= PERT_TOL, (pe, sc)
        worst["rho'"], worst["p'"] = pe
    return worst


def test_cfg2_full_128_all_100_steps():
    """BASELINE.json configs[1] exactly: 128^3, 100 steps, against the full-grid oracle (about half a minute of CPU)"""
    w = W.make(2)
    r = _run_pair(w, w.steps)
    assert max(r[1][0].values()) <= ONE_STEP, r[1][0]
    assert max(r[w.steps][0].values()) <= MULTI_STEP, r[w.steps][0]
    assert r["cons0"].max() <= CONS and r["cons1"].max() <= CONS


def test_cfg2_full_128_windows():
    n = 128
    _window_check(2, 2, [((64, 64, 64), 24), ((64, 64, 77), 24), ((10, 64, 4), 24), ((64, 120, 124), 24)])


def test_cfg3_full_256_all_50_steps_L1():
    """BASELINE.json configs[2] exactly: 256^3, 50 steps, against the full-grid oracle (the 200-cell apron of a window
    would cover the grid anyway; about 2.5 minutes of oracle time on the GPU box's host cores)"""
    w = W.make(3)
    r = _run_pair(w, w.steps)
    assert max(r[1][1].values()) <= L1_SHOCK, r[1][1]
    assert max(r[w.steps][1].values()) <= L1_SHOCK, r[w.steps][1]
    assert r["cons1"].max() <= CONS
    print("cfg3 256^3 x 50 steps: L1", r[w.steps][1], "max", r[w.steps][0])


def test_cfg3_full_256_windows_L1():
    _window_check(3, 2, [((128, 128, 128), 32), ((128, 128, 100), 24), ((8, 8, 8), 24)], tol=L1_SHOCK, norm="l1")


def test_cfg4_full_512_windows():
    c = 256
    r45 = int(0.45 * 512)
    _window_check(4, 2, [((c, c, c), 24), ((c + 170, c, c), 24), ((c, c + r45, c), 24), ((c, c, c + int(0.48 * 512)), 24),
                         ((c, 6, c), 24), ((6, 6, 6), 24)])


def test_cfg4_full_512_all_20_steps_window():
    """the headline config at its full size AND its full step count (BASELINE.json configs[3]: 512^3, 20 steps), in the
    launch configuration bench.py times: one 32^3 window in the convective shell, oracle on the window plus its
    80-cell apron (192^3 cells, 20 steps)."""
    c = 256
    _window_check(4, 20, [((c + 175, c, c), 32)], tol=MULTI_STEP)


@pytest.mark.skipif(not torch.cuda.is_available() or torch.cuda.get_device_properties(0).total_memory < 150e9,
                    reason="1024^3 needs ~129 GB of HBM")
def test_cfg5_full_1024_windows_all_5_steps():
    """BASELINE.json configs[4]: 1024^3, all of its 5 steps; windows in the core, the shell, the FV edge and a corner"""
    c = 512
    _window_check(5, 5, [((c, c, c), 24), ((c + 340, c, c), 24), ((c, c + int(0.45 * 1024), c), 24), ((6, 6, 6), 24)], nzs_load=8,
                  tol=MULTI_STEP)
