"""Pins of the oracle's boundary source (43a-d), that do NOT re-type its formula.

What the paper fixes about the focused / packet source and what each test would catch.  Every mutation named in a
docstring below was applied to a copy of oracle/fvnl_oracle.cpp and the test confirmed to fail under it, and every one
of the 12 mutations tried (signs, exchanged components, normalisation, curvature sign / factor / absence, origin of x2,
envelope exponent -10 / 2, |x2|, inward normals of x-hi and y-hi) fails at least one test (A13, A14):

  geometry   (43b,c): (q2, q3) = g (F, -x2)/sqrt(x2^2 + F^2) -- a vector of length |g| = |q1 - 1| (43a) that points from
             the aperture point (0, x2) to the focus (F, 0) while the medium is compressed.
  phase      tau = t + x2^2/(2F): the rim of the aperture fires EARLIER than its centre, so that the
             wavelets meet at the focus.
  envelope   (43d) with "t = 0 when the center of the packet was precisely on the left border" and "t0 ... chosen for
             the packet to be numerically zero at machine precision": a packet that is flat around
             tau = 0 and vanishes for large |tau| -- reading A13, exp(-(tau/4)^10), against the printed exponent -10.
  plane limit F -> infinity of (43) is the plane piston that the Fubini pin (P6) already fixes.
"""
import math

import numpy as np
import pytest

import workloads as W
from oracle.oracle import Oracle, EXTRAP, SOURCE, XLO, XHI, YLO, YHI, SINE, PACKET

DX = W.LAMBDA_1MHZ / 16
FREQ = 1.0e6


def source(shape=PACKET, amp=3e-4, focus_cells=96.0, centre_cells=80.0, aperture_cells=64.0, tau0=0.0):
    return dict(shape=shape, amp=amp, freq_hz=FREQ, focus_m=focus_cells * DX, centre_m=centre_cells * DX,
                half_aperture_m=aperture_cells * DX, t0_s=tau0 / FREQ, steep=0.0)


def oracle_with(side, src, nx=160, ny=160, threads=0):
    o = Oracle(nx, ny, DX, DX, **W.MEDIUM_WATER, threads=threads)
    o.set_bc(side, SOURCE, src)
    return o


# inward unit normal n and "along the edge" unit vector e (the direction in which `along` grows) of every side, in (x, y)
SIDES = {XLO: ((1.0, 0.0), (0.0, 1.0)), XHI: ((-1.0, 0.0), (0.0, 1.0)),
         YLO: ((0.0, 1.0), (1.0, 0.0)), YHI: ((0.0, -1.0), (1.0, 0.0))}


@pytest.mark.parametrize("side", [XLO, XHI, YLO, YHI])
def test_momentum_has_length_g_and_points_at_the_focus(side):
    """(43a-c).  On every aperture cell of every side: |(q2, q3)| = |q1 - 1| (cos^2 + sin^2 = 1 pins
    the normalisation by sqrt(x2^2 + F^2)), and the momentum is parallel to the ray from the aperture point to the focus,
    which lies at distance F along the inward normal from the aperture centre, pointing AT it when q1 > 1.
    Fails under: along-edge component with the wrong sign (momentum points away from the axis); q2 / q3 exchanged;
    normalisation by F instead of sqrt(x2^2 + F^2); a side whose normal component is not turned inwards."""
    src = source()
    o = oracle_with(side, src)
    n, e = SIDES[side]
    F, c = src["focus_m"], src["centre_m"]
    seen_pos = seen_neg = 0
    for t in (0.13e-6, 0.4e-6, 0.71e-6, 1.9e-6):
        for cell in range(0, 160, 3):
            along = (cell + 0.5) * DX
            inside, q = o.source_cell(side, along, 0.0, t)
            d = along - c
            assert inside == (abs(d) <= src["half_aperture_m"])
            if not inside:
                continue
            g = q[0] - 1.0
            mom = np.array([q[1], q[2]])
            assert np.hypot(*mom) == pytest.approx(abs(g), rel=1e-13, abs=2.3e-16)   # q1 = 1 + g is rounded at ulp(1)
            ray = np.array([F * n[0] - d * e[0], F * n[1] - d * e[1]])           # aperture point -> focus
            cross = mom[0] * ray[1] - mom[1] * ray[0]
            assert abs(cross) <= 1e-15 * np.hypot(*mom) * np.hypot(*ray)
            if abs(g) > 1e-9:
                assert np.sign(mom @ ray) == np.sign(g)
                seen_pos += g > 0
                seen_neg += g < 0
    assert seen_pos > 20 and seen_neg > 20


def test_rim_fires_before_the_centre():
    """tau = t + x2^2/(2F): a point of the aperture at distance x2 from the axis runs AHEAD of the centre by
    x2^2/(2 F lambda) periods, i.e. its signal at time t equals the centre's signal at the LATER time t + x2^2/(2 F c0)
    (same g; pinned through q1 = 1 + g only, so that no momentum formula enters).
    Fails under: tau = t - x2^2/(2F) (a defocusing aperture); x2^2/F without the 1/2; d measured from the edge's corner."""
    src = source(shape=PACKET, tau0=-1.0)
    o = oracle_with(XLO, src)
    F, c0 = src["focus_m"], W.MEDIUM_WATER["c0"]
    for cells_off in (10.0, 33.0, 60.0):
        d = cells_off * DX
        lead = d * d / (2.0 * F * c0)                                            # seconds
        for t in (0.2e-6, 0.9e-6, 1.45e-6):
            _, q_rim = o.source_cell(XLO, src["centre_m"] + d, 0.0, t)
            _, q_mirror = o.source_cell(XLO, src["centre_m"] - d, 0.0, t)
            _, q_centre_later = o.source_cell(XLO, src["centre_m"], 0.0, t + lead)
            assert q_rim[0] - 1.0 == pytest.approx(q_centre_later[0] - 1.0, rel=1e-9, abs=1e-16)
            assert q_rim[0] == q_mirror[0]                                       # even in x2
    # and it matters: half a period of lead at x2 = sqrt(F lambda)
    d = math.sqrt(F * W.LAMBDA_1MHZ)
    _, a = o.source_cell(XLO, src["centre_m"] + d, 0.0, 1.25e-6)                 # centre at tau = 0.25: crest
    _, b = o.source_cell(XLO, src["centre_m"], 0.0, 1.25e-6)
    assert (a[0] - 1.0) == pytest.approx(-(b[0] - 1.0), rel=1e-3)


def test_packet_envelope_against_the_papers_description():
    """(43d) + PAPER.md:287.  The paper prints the envelope as e^{-(tau/4)^{-10}}, which is 0 at tau = 0 and 1 for large
    |tau| -- not a packet.  The text fixes what it must be: "t = 0 when the center of the packet was precisely on the left
    border" (the envelope is centred on, and largest at, tau = 0) and "the value of t0 was chosen for the packet to be
    numerically zero at machine precision" (it vanishes for large |tau|); "wave packets".  Reading A13:
    exp(-(tau/4)^10), a flat packet of about 8 periods.
    Fails under: the printed exponent -10 (crest at tau = 1/4 would be 0, tail would be full amplitude); exponent 2
    (Gaussian: not flat, 0.94 instead of 1 - 1e-6 at tau = 1); tau/4 replaced by tau or tau/8; missing carrier sin(2 pi tau)."""
    amp = 3e-4
    src = source(shape=PACKET, amp=amp, focus_cells=0.0, aperture_cells=0.0)      # plane: tau = f t
    o = oracle_with(XLO, src)

    def g(tau):
        inside, q = o.source_cell(XLO, 50 * DX, 0.0, tau / FREQ)
        assert inside
        return q[0] - 1.0

    # centred on tau = 0, odd carrier, crests of full amplitude near the centre
    assert g(0.0) == 0.0
    for tau in (0.25, 1.25, 2.25):
        assert g(tau) == pytest.approx(-g(-tau), rel=1e-12)
    assert g(0.25) == pytest.approx(amp, rel=1e-9)                                # flat top: 1 - (1/16)^10
    assert g(1.25) == pytest.approx(amp, rel=1e-4)                                # (1.25/4)^10 = 9e-6
    assert g(-0.75) == pytest.approx(amp, rel=1e-6)
    # crest amplitudes decrease monotonically away from the centre and the packet is "about 8 periods" long
    crests = [abs(g(k + 0.25)) for k in range(0, 8)]
    assert all(a > b for a, b in zip(crests[:6], crests[1:6])) and crests[6] <= crests[5] and crests[7] <= crests[6]
    assert crests[2] > 0.99 * amp and crests[3] > 0.85 * amp and crests[4] < 0.2 * amp and crests[5] < 1e-5 * amp
    # numerically zero at machine precision: beyond 5.8 periods the packet is below one ulp of the unit background
    for tau in (5.85, 6.25, 7.25, 9.125, 20.25, -5.85, -6.25, -9.125):
        assert abs(g(tau)) < 2.3e-16
    # C4's own t0 (workloads.c4_hifu): zero on the whole aperture at t = 0, as PAPER.md:287 demands
    w = W.c4_hifu()
    s4 = w.bc[0][1]
    o4 = Oracle(64, w.ny, w.dx, w.dy, **w.medium)
    o4.set_bc(XLO, SOURCE, s4)
    for j in range(0, w.ny, 16):
        inside, q = o4.source_cell(XLO, (j + 0.5) * w.dy, 0.0, 0.0)
        if inside:
            assert abs(q[0] - 1.0) < 1e-24 and abs(q[1]) < 1e-24 and abs(q[2]) < 1e-24


def test_infinite_focus_is_the_plane_piston():
    """F -> infinity in (43): x2^2/(2F) -> 0, F/sqrt(x2^2 + F^2) -> 1, x2/sqrt(...) -> 0: the plane piston q = (1 + g, g, 0)
    (reading A16), whose amplitude and nonlinear distortion the Fubini pin (P6, test_oracle_pins.py) fixes.  The oracle's
    focused branch at F = 1e12 m must reproduce its own plane branch (focus_m <= 0) to round-off.
    Fails under: any dimensional slip in the curvature term (e.g. d^2/(2 F) without 1/lambda stays visible at 1e12 only if
    mis-scaled by >= 1e9, so this is the weakest of the pins) and under a normal component that is not g cos(theta)."""
    for shape in (SINE, PACKET):
        far = oracle_with(XLO, source(shape=shape, focus_cells=1e12 / DX, tau0=0.3))
        plane = oracle_with(XLO, source(shape=shape, focus_cells=0.0, tau0=0.3))
        for cell in (20, 80, 131):
            for t in (0.1e-6, 0.77e-6, 2.4e-6):
                a, qa = far.source_cell(XLO, (cell + 0.5) * DX, 0.0, t)
                b, qb = plane.source_cell(XLO, (cell + 0.5) * DX, 0.0, t)
                assert a and b
                assert qa[0] == pytest.approx(qb[0], abs=2.3e-16)
                assert qa[1] == pytest.approx(qb[1], rel=1e-12)                   # x2^2/(2 F lambda) <= 1e-14 periods
                assert qb[1] == pytest.approx(qb[0] - 1.0, abs=2.3e-16)           # A16: q2 = g
                assert abs(qa[2]) <= 1e-13 * abs(qb[1]) and qb[2] == 0.0


@pytest.fixture(scope="module")
def focused_cw_run():
    """A small LINEAR run of the oracle alone: continuous focused SINE source (amp 1e-6) on x-lo, F = 96 cells = 6 lambda,
    half-aperture 64 cells = 4 lambda, 160 x 160 cells, extrapolation elsewhere; 280 steps to a periodic state, then the
    time-maximum of |q1 - 1| on the axis over 40 steps (two periods)."""
    amp = 1e-6
    o = oracle_with(XLO, source(shape=SINE, amp=amp))
    assert o.step(280, 0.8, 1) == 0
    axis_max = np.zeros(160)
    for _ in range(40):
        assert o.step(1, 0.8, 1) == 0
        q1 = o.get_state()[0]
        axis_max = np.maximum(axis_max, np.abs(0.5 * (q1[79] + q1[80]) - 1.0))   # aperture centre = boundary of rows 79|80
    return amp, axis_max, o.get_state()


def test_focused_source_focuses(focused_cw_run):
    """Physics of (43) as a whole ("a transducer with the shape of a circle arc produces a focusing wave"):
    the on-axis pressure amplitude of the linear field rises from the source towards the focus, peaks a little before the
    geometric focus (the focal shift of an aperture of Fresnel number a^2/(lambda F) = 2.7) and clearly exceeds the source
    amplitude.
    Fails under: tau = t - x2^2/(2F) (the beam diverges: the on-axis maximum sits at the source); a missing curvature
    term (plane piston: no gain); x2^2/F without the 1/2; q2 / q3 exchanged; x2 measured from the corner of the edge."""
    amp, axis_max, _ = focused_cw_run
    F = 96
    peak = int(axis_max.argmax())
    assert 0.75 * F <= peak <= 1.05 * F, peak
    assert axis_max[peak] > 2.5 * amp
    assert axis_max[peak] > 1.8 * axis_max[:F // 3].max()
    assert axis_max[150] < 0.6 * axis_max[peak]                                  # and it spreads again behind the focus


def test_focused_field_is_mirror_symmetric_about_the_axis(focused_cw_run):
    """The arc is symmetric about x2 = 0 (and the paper computes only the upper half): q1 and
    q2 even, q3 odd about the aperture axis, to round-off.
    Fails under: d measured from a wrong centre; a q3 that is even in x2 (e.g. |x2| in (43c))."""
    amp, _, q = focused_cw_run
    q1, q2, q3 = q
    assert np.abs(q1 - q1[::-1]).max() <= 1e-12 * amp
    assert np.abs(q2 - q2[::-1]).max() <= 1e-12 * amp
    assert np.abs(q3 + q3[::-1]).max() <= 1e-12 * amp
    assert np.abs(q3).max() > 0.2 * amp


def _load_c4_script():
    import importlib.util
    import os
    spec = importlib.util.spec_from_file_location(
        "make_c4_windows", os.path.join(os.path.dirname(__file__), "golden", "make_c4_windows.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


def test_c4_golden_script_round_trip(tmp_path):
    """tests/golden/make_c4_windows.py on a scaled-down C4: what it writes is, bit for bit, what the oracle holds (hex
    floats), so neither the script nor the file format can go stale; the stored statistics are those of the state."""
    mod = _load_c4_script()
    w = W.c4_hifu(nx=160, ny=96, steps=60, focus_cells=60.0, aperture_cells=30.0, tau0=-1.0)
    lines = mod.run(w, (20, 60), 6, 0)
    path = tmp_path / "c4_small.txt"
    path.write_text(mod.HEADER + "\n".join(lines) + "\n")
    gold = mod.read(str(path))
    assert gold["config"]["steps"] == [20, 60] and gold["config"]["win"] == 6
    o = Oracle(w.nx, w.ny, w.dx, w.dy, **w.medium, threads=0)
    o.set_bc(XLO, SOURCE, w.bc[0][1])
    assert o.step(20, w.value, 1) == 0 and o.step(40, w.value, 1) == 0
    q = o.get_state()
    cp = gold["checkpoints"][60]
    assert cp["t"] == o.info()["t"] and cp["M"] == o.info()["M"]
    assert set(cp["windows"]) == {"edge_axis", "edge_half_aperture", "focus", "peak_q1", "peak_q3"}
    for wd in cp["windows"].values():
        for m in range(3):
            assert np.array_equal(wd["q"][m], q[m][wd["j0"]:wd["j0"] + 6, wd["i0"]:wd["i0"] + 6])
    assert cp["stats"][0]["max"] == np.abs(q[0] - 1.0).max() and cp["stats"][2]["l1"] == np.abs(q[2]).sum()


def test_c4_golden_file_is_the_full_config():
    """The stored file (when present) is C4 of BASELINE.json at full size and full step count, and what it holds is a
    focused packet: nothing on the aperture at t = 0 ... the field at the focus exceeds the source amplitude (focusing
    gain), the source edge is silent again once the packet has left, q3 is odd about the axis."""
    import os
    mod = _load_c4_script()
    if not os.path.exists(mod.OUT):
        pytest.skip("tests/golden/c4_full_windows.txt not generated yet")
    gold = mod.read()
    w = W.c4_hifu()
    cfg = gold["config"]
    assert (cfg["nx"], cfg["ny"], cfg["nu_w"], cfg["steps"][-1]) == (8192, 2048, 0.8, 4000) == (w.nx, w.ny, w.value, w.steps)
    amp = w.bc[0][1]["amp"]
    cps = gold["checkpoints"]
    for cp in cps.values():
        assert abs(cp["cfl"] - 0.8) < 2.5e-4 * 4                       # paper: std of nu <= 2.5e-4 on HIFU
    assert 0.9 * amp < cps[400]["stats"][0]["max"] < 1.5 * amp          # packet being emitted
    if 4000 not in cps:                                                 # (a file copied from the script's .partial output)
        return
    assert cps[3000]["stats"][0]["max"] > 2.0 * amp                     # at the focus (step ~2925): focusing gain
    assert np.abs(cps[4000]["windows"]["edge_axis"]["q"][0] - 1.0).max() < 1e-3 * amp
    ax = cps[3000]["windows"]["focus"]                                  # window centred on the axis: rows j0 .. j0+19
    assert ax["j0"] + 10 == w.ny // 2
    assert np.abs(ax["q"][2] + ax["q"][2][::-1]).max() <= 1e-9 * np.abs(ax["q"][2]).max()


def test_c4_sensitivity_file_is_consistent_with_the_golden_file():
    """tests/golden/c4_sensitivity.txt (when present): the oracle compiled with FMA contraction against the standard oracle's
    stored C4 run -- written by tests/golden/make_c4_sensitivity.py, oracle only.  Its checkpoints are checkpoints of the
    golden file, every window of the golden file has its three fields, 'worst' is the maximum of the step's windows, and at
    the first checkpoint (packet still being emitted) the two roundings agree to far better than the parity bar."""
    import os
    mod = _load_c4_script()
    path = os.path.join(os.path.dirname(mod.OUT), "c4_sensitivity.txt")
    if not (os.path.exists(path) and os.path.exists(mod.OUT)):
        pytest.skip("tests/golden/c4_sensitivity.txt not generated yet")
    gold = mod.read()
    windows, worst = {}, {}
    for line in open(path):
        if line.startswith("window"):
            _, cp, name, m, v = line.split()
            windows.setdefault(int(cp), {})[(name, int(m))] = float(v)
        elif line.startswith("worst"):
            worst[int(line.split()[1])] = float(line.split()[2])
    assert worst and set(worst) == set(windows)
    for cp, d in windows.items():
        assert cp in gold["checkpoints"]
        assert set(d) == {(name, m) for name in gold["checkpoints"][cp]["windows"] for m in range(3)}
        assert worst[cp] == pytest.approx(max(d.values()), rel=1e-3)
    assert worst[min(worst)] < 1e-10
