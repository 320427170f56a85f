"""Pins P1-P16 (DESIGN.md / SURVEY.md 8(c)): the float64 oracle checked against what the paper's
definition and the mathematics fix -- never against itself and never against the CUDA path."""
import numpy as np
import pytest
import scipy.signal

from paper_1605_07023_b200 import synth

N, S, O, W = 32, 5, 4, 3


def centre_const(n, s, o):
    # expected (cell, row) for u = 0: the sample sits on cell floor(n/2) (FFT-centre convention)
    # nearest S cells start at ceil(n/2 - s/2)
    return int(np.ceil(n // 2 - s / 2.0))


def rand_kernel(rng, w=W, o=O, s=S):
    return (rng.standard_normal((w, o, s)) + 1j * rng.standard_normal((w, o, s))).astype(np.complex64)


def brute_gather(n, s, o, w, p, uvw, vis, weights, kernel):
    """P4: independent pure-Python gather form.  For every cell loop over all samples."""
    import math
    out = np.zeros((n, n, p), dtype=np.complex128)
    nv = uvw.shape[0]
    pos = []
    for k in range(nv):
        u, v, ww = (float(x) for x in uvw[k])
        # position in oversampled units, rounded half up; footprint start by the ceil rule
        pu = math.floor((u + n // 2) * o + 0.5)
        pv = math.floor((v + n // 2) * o + 0.5)
        # the S cells c with d = c - pu/o in (-s/2, s/2]:  first one is floor(pu/o - s/2) + 1
        i0 = (2 * pu - s * o) // (2 * o) + 1
        j0 = (2 * pv - s * o) // (2 * o) + 1
        # row: cell i0 lies at d = -s/2 + 1 - su/o  =>  su = pu - o*s/2 + o - i0*o   (o*s even or o == 1)
        assert (o * s) % 2 == 0 or o == 1
        su = 0 if o == 1 else pu - (o * s) // 2 + o - i0 * o
        sv = 0 if o == 1 else pv - (o * s) // 2 + o - j0 * o
        assert 0 <= su < o and 0 <= sv < o
        plane = min(int(math.floor(abs(ww))), w - 1)
        pos.append((i0, j0, su, sv, plane))
    for j in range(n):
        for i in range(n):
            for k in range(nv):
                i0, j0, su, sv, plane = pos[k]
                if i0 < 0 or i0 + s > n or j0 < 0 or j0 + s > n:
                    continue
                if 0 <= i - i0 < s and 0 <= j - j0 < s:
                    g = complex(kernel[plane, sv, j - j0]) * complex(kernel[plane, su, i - i0])
                    for q in range(p):
                        out[j, i, q] += float(weights[k]) * complex(vis[k, q]) * g
    return out


def test_p1_single_unit_visibility(oracle_mod):
    rng = np.random.default_rng(1)
    kernel = rand_kernel(rng)
    # u = 3 + 1/4 cells, v = -2 + 2/4 cells from the centre; plane 1
    uvw = np.array([[3.25, -1.5, 1.2]], dtype=np.float32)
    vis = np.ones((1, 1), dtype=np.complex64)
    g = oracle_mod.grid(N, S, O, W, 1, uvw, vis, np.ones(1, np.float32), kernel)
    # by hand: position 16+3.25 = 19.25 -> cells within (-2.5, 2.5] of it: 17..21; tap t at d = t-1.5-su/4 from
    # the sample; cell 17 is at 17-19.25 = -2.25 = 0 - 1.5 - 3/4 -> su = 3
    i0, su = 17, 3
    # v: 16-1.5 = 14.5 -> cells within (-2.5, 2.5]: 13..17 (12 is at exactly -2.5: excluded);
    # cell 13 at -1.5 = 0 - 1.5 - 0/4 -> sv = 0
    j0, sv = 13, 0
    expect = np.zeros((N, N), dtype=np.complex128)
    expect[j0:j0 + S, i0:i0 + S] = np.outer(kernel[1, sv].astype(np.complex128),
                                           kernel[1, su].astype(np.complex128))
    np.testing.assert_allclose(g[:, :, 0], expect, rtol=0, atol=1e-15)
    assert np.count_nonzero(g) == S * S


def test_p1_rows_cols_not_transposed_and_no_conjugate(oracle_mod):
    kernel = np.zeros((1, 1, 3), dtype=np.complex64)
    kernel[0, 0] = [1 + 2j, 3 + 0j, 0 + 5j]
    uvw = np.array([[2.0, -4.0, 0.0]], dtype=np.float32)    # u -> column, v -> row
    vis = np.array([[1j]], dtype=np.complex64)
    g = oracle_mod.grid(16, 3, 1, 1, 1, uvw, vis, np.array([2.0], np.float32), kernel)[:, :, 0]
    # centre 8: u=2 -> col 10, taps at cols 9..11 ; v=-4 -> row 4, rows 3..5  (ceil(x+8-1.5))
    k = kernel[0, 0].astype(np.complex128)
    assert g[3, 9] == 2.0 * 1j * k[0] * k[0]
    assert g[5, 9] == 2.0 * 1j * k[2] * k[0]     # row index uses the v taps
    assert g[3, 11] == 2.0 * 1j * k[0] * k[2]
    assert g[4, 10] == 2.0 * 1j * k[1] * k[1]
    assert np.count_nonzero(g) == 9


@pytest.mark.parametrize("P", [1, 4])
def test_p2_linearity(oracle_mod, P):
    uvw, vis1, wts, kernel = synth.random_problem(2, 500, N, S, O, W, P, spread=0.3)
    _, vis2, _, _ = synth.random_problem(3, 500, N, S, O, W, P, spread=0.3)
    a, b = np.float32(0.5), np.float32(-2.0)        # exact in fp32 so inputs combine exactly enough
    comb = (a * vis1 + b * vis2).astype(np.complex64)
    g1 = oracle_mod.grid(N, S, O, W, P, uvw, vis1, wts, kernel)
    g2 = oracle_mod.grid(N, S, O, W, P, uvw, vis2, wts, kernel)
    gc = oracle_mod.grid(N, S, O, W, P, uvw, comb, wts, kernel)
    # comb is rounded to fp32; compare against the same rounded values promoted
    exact = float(a) * g1 + float(b) * g2
    comb_err = np.abs(comb.astype(np.complex128) - (float(a) * vis1.astype(np.complex128)
                                                    + float(b) * vis2.astype(np.complex128))).max()
    assert comb_err < 1e-6
    scale = np.abs(exact).max()
    assert np.abs(gc - exact).max() <= 1e-12 * scale + 500 * comb_err * 4 * 4


@pytest.mark.parametrize("P", [1, 4])
def test_p3_grid_sum(oracle_mod, P):
    uvw, vis, wts, kernel = synth.random_problem(4, 2000, N, S, O, W, P, spread=0.55)
    q = oracle_mod.quantise(N, S, O, W, uvw)
    assert 0 < q["valid"].sum() < len(q["valid"])     # some samples fall off the edge
    g = oracle_mod.grid(N, S, O, W, P, uvw, vis, wts, kernel)
    ksum = kernel.astype(np.complex128).sum(axis=2)           # [W][O]
    expect = np.zeros(P, dtype=np.complex128)
    for n in np.nonzero(q["valid"])[0]:
        expect += (float(wts[n]) * vis[n].astype(np.complex128)
                   * ksum[q["wp"][n], q["sv"][n]] * ksum[q["wp"][n], q["su"][n]])
    np.testing.assert_allclose(g.sum(axis=(0, 1)), expect, rtol=1e-11, atol=1e-11)


@pytest.mark.parametrize("s,o,P", [(5, 4, 1), (4, 3, 2), (1, 1, 1), (8, 8, 4)])
def test_p4_brute_force_gather(oracle_mod, s, o, P):
    n, w = 24, 2
    uvw, vis, wts, kernel = synth.random_problem(5 + s, 60, n, s, o, w, P, spread=0.6)
    g = oracle_mod.grid(n, s, o, w, P, uvw, vis, wts, kernel)
    ref = brute_gather(n, s, o, w, P, uvw, vis, wts, kernel)
    assert np.abs(ref).max() > 0
    np.testing.assert_allclose(g, ref, rtol=1e-13, atol=1e-13)


def test_p5_suboffset_sweep_and_tie_break(oracle_mod):
    n, s, o = 64, 6, 8
    # even S: at su = 0 the taps sit at d = -2..3, so a sample on cell 32 starts at cell 30
    base = 0.0
    us = []
    for k in range(o):
        us.append(base + k / o)                 # exactly on oversampled point k
    for k in range(o - 1):
        us.append(base + (k + 0.5) / o)         # tie: half up -> k+1
    us.append(base + (o - 0.5) / o)             # tie at the last point: next cell, row 0
    us.append(-0.5 / o)                         # negative tie: half up -> position 0
    us.append(-1.5 / o)                         # -> position -1/o: previous cell
    uvw = np.zeros((len(us), 3), dtype=np.float32)
    uvw[:, 0] = us
    assert np.all(uvw[:, 0].astype(np.float64) == np.array(us))     # exactly representable
    q = oracle_mod.quantise(n, s, o, 1, uvw)
    # rounded position p (oversampled units relative to cell 32).  Cell i0 lies at
    # d = -s/2 + 1 - su/o = -2 - su/o from it:  i0*o + su = 30*o + p
    def expect(p):
        return 30 + p // o, p % o
    ps = list(range(o)) + [k + 1 for k in range(o - 1)] + [o, 0, -1]
    for idx, p in enumerate(ps):
        c, su = expect(p)
        assert (q["i0"][idx], q["su"][idx]) == (c, su), (idx, p, q["i0"][idx], q["su"][idx], c, su)
    assert np.all(q["j0"] == 30) and np.all(q["sv"] == 0) and np.all(q["valid"] == 1)
    # u = 0 exactly: cells 30..35 (d = -2..3), row 0; u = 1/o: same cells, row 1;
    # u = -1.5/o -> position -1/o: cells 29..34, row o-1
    assert (q["i0"][0], q["su"][0]) == (30, 0)
    assert (q["i0"][1], q["su"][1]) == (30, 1)
    assert (q["i0"][-1], q["su"][-1]) == (29, o - 1)


def test_p5_odd_support_centre(oracle_mod):
    # odd S: a sample exactly on a cell has its centre tap (t = (S-1)/2) at d = 0 only if
    # d = t - S/2 + 1 - su/O = 0 -> su = O/2; cells start at ceil(16 - 2.5) = 14
    q = oracle_mod.quantise(32, 5, 4, 1, np.zeros((1, 3), np.float32))
    assert (q["i0"][0], q["su"][0]) == (14, 2)
    assert q["i0"][0] == centre_const(32, 5, 4)


def test_p6_whole_cell_translation(oracle_mod):
    uvw, vis, wts, kernel = synth.random_problem(6, 400, 48, S, O, W, 2, spread=0.3)
    uvw = np.round(uvw * 64) / 64            # keeps u+1 exact in fp32
    uvw = uvw.astype(np.float32)
    g0 = oracle_mod.grid(48, S, O, W, 2, uvw, vis, wts, kernel)
    sh = uvw.copy()
    sh[:, 0] += 1.0
    sh[:, 1] -= 2.0
    g1 = oracle_mod.grid(48, S, O, W, 2, sh, vis, wts, kernel)
    assert np.array_equal(g1[:-2, 1:], g0[2:, :-1])       # bit-for-bit
    # what slid in from outside the grid is empty: column 0 (u + 1) and the last two rows (v - 2)
    assert np.count_nonzero(g1[:, 0]) == 0 and np.count_nonzero(g1[-2:, :]) == 0
    # and nothing was lost at the far edges of the original
    assert np.count_nonzero(g0[:, -1]) == 0 and np.count_nonzero(g0[:2, :]) == 0


@pytest.mark.parametrize("P", [1, 4])
def test_p7_adjoint_identity(oracle_mod, P):
    rng = np.random.default_rng(7)
    uvw, vis, wts, kernel = synth.random_problem(7, 300, N, S, O, W, P, spread=0.55)
    G = rng.standard_normal((N, N, P)) + 1j * rng.standard_normal((N, N, P))
    gv = oracle_mod.grid(N, S, O, W, P, uvw, vis, wts, kernel)
    dg = oracle_mod.degrid(N, S, O, W, P, uvw, wts, kernel, G)
    lhs = np.vdot(gv, G)                       # sum conj(grid(V)) * G
    rhs = np.vdot(vis.astype(np.complex128), dg)
    assert abs(lhs - rhs) <= 1e-12 * abs(lhs)


def test_p8_box_filter_of_histogram(oracle_mod):
    n, s = 40, 4
    uvw, vis, wts, _ = synth.random_problem(8, 3000, n, s, 1, 1, 1, spread=0.4)
    kernel = np.ones((1, 1, s), dtype=np.complex64)
    g = oracle_mod.grid(n, s, 1, 1, 1, uvw, vis, wts, kernel)[:, :, 0]
    # nearest cell (half up) by numpy; S=4,O=1: cells start at nearest - 1 (d = -1..2)
    col = np.floor(uvw[:, 0].astype(np.float64) + n // 2 + 0.5).astype(int)
    row = np.floor(uvw[:, 1].astype(np.float64) + n // 2 + 0.5).astype(int)
    hist = np.zeros((n, n), dtype=np.complex128)
    np.add.at(hist, (row, col), wts.astype(np.float64) * vis[:, 0].astype(np.complex128))
    box = scipy.signal.convolve2d(hist, np.ones((s, s)), mode="full")
    # full conv index m = cell + t ; footprint cells = nearest-1 .. nearest+2 -> shift by 1
    expect = box[1:1 + n, 1:1 + n]
    np.testing.assert_allclose(g, expect, rtol=1e-12, atol=1e-12)


def test_p9_nearest_cell_histogram(oracle_mod):
    n = 32
    uvw, vis, wts, _ = synth.random_problem(9, 2000, n, 1, 1, 1, 1, spread=0.49)
    g = oracle_mod.grid(n, 1, 1, 1, 1, uvw, vis, wts, np.ones((1, 1, 1), np.complex64))[:, :, 0]
    col = np.floor(uvw[:, 0].astype(np.float64) + n // 2 + 0.5).astype(int)
    row = np.floor(uvw[:, 1].astype(np.float64) + n // 2 + 0.5).astype(int)
    hist = np.zeros((n, n), dtype=np.complex128)
    ok = (row >= 0) & (row < n) & (col >= 0) & (col < n)
    np.add.at(hist, (row[ok], col[ok]), (wts.astype(np.float64) * vis[:, 0].astype(np.complex128))[ok])
    np.testing.assert_allclose(g, hist, rtol=1e-13, atol=1e-13)


def test_p10_compression_invariance(oracle_mod):
    # samples with the same oversampled position may be summed first
    uvw, vis, wts, kernel = synth.random_problem(10, 600, N, S, O, W, 2, spread=0.3)
    uvw = np.repeat(uvw[:200], 3, axis=0)              # triples share a position exactly
    q = oracle_mod.quantise(N, S, O, W, uvw)
    g = oracle_mod.grid(N, S, O, W, 2, uvw, vis, wts, kernel)
    merged_v = (wts[:, None].astype(np.float64) * vis.astype(np.complex128)).reshape(200, 3, 2).sum(1)
    # merged values are not fp32-representable in general: apply them through linearity, i.e.
    # grid three unit-weight runs of the de-duplicated positions and add (all in float64)
    g_m = np.zeros_like(g)
    for r in range(3):
        g_m += oracle_mod.grid(N, S, O, W, 2, uvw[r::3], vis[r::3], wts[r::3], kernel)
    np.testing.assert_allclose(g, g_m, rtol=1e-12, atol=1e-12)
    # and the sum of a group equals its merged value times the plane sums (ties compression to P3)
    ksum = kernel.astype(np.complex128).sum(axis=2)
    idx = np.arange(0, 600, 3)
    expect = (merged_v * (ksum[q["wp"][idx], q["sv"][idx]] * ksum[q["wp"][idx], q["su"][idx]])[:, None]
              * q["valid"][idx][:, None]).sum(0)
    np.testing.assert_allclose(g.sum((0, 1)), expect, rtol=1e-11)


def test_p11_permutation_invariance(oracle_mod):
    uvw, vis, wts, kernel = synth.random_problem(11, 800, N, S, O, W, 4, spread=0.4)
    g = oracle_mod.grid(N, S, O, W, 4, uvw, vis, wts, kernel)
    perm = np.random.default_rng(0).permutation(800)
    gp = oracle_mod.grid(N, S, O, W, 4, uvw[perm], vis[perm], wts[perm], kernel)
    np.testing.assert_allclose(gp, g, rtol=0, atol=1e-12 * np.abs(g).max())


def test_p12_w_plane_selection(oracle_mod):
    ws = np.array([0.0, 0.5, 0.999, 1.0, 1.5, -1.5, 2.0, 2.5, 3.0, 7.0, -9.0, 1e30], dtype=np.float32)
    uvw = np.zeros((len(ws), 3), dtype=np.float32)
    uvw[:, 2] = ws
    q = oracle_mod.quantise(N, S, O, 3, uvw)
    assert list(q["wp"]) == [0, 0, 0, 1, 1, 1, 2, 2, 2, 2, 2, 2]
    assert np.all(q["valid"] == 1)


def test_p13_edges_and_nonfinite(oracle_mod):
    n, s, o = 16, 4, 2
    kernel = np.ones((1, o, s), dtype=np.complex64)
    # S=4: u=0 -> cells 7..10.  i0 = 0 <=> u in [-7, -6.5] ; i0 + S = N <=> i0 = 12 <=> u in [5, 5.5]
    # (rounded to the nearest 1/2): u = 5.5 is the last valid position, u = 6 the first invalid one
    uvw = np.array([[-7.0, 0, 0], [5.5, 0, 0], [-7.5, 0, 0], [6.0, 0, 0], [0, -8.0, 0], [0, 6.0, 0],
                    [np.nan, 0, 0], [0, np.inf, 0], [0, 0, np.nan], [1e30, 0, 0], [-1e30, 0, 0],
                    [0, 0, -np.inf]], dtype=np.float32)
    q = oracle_mod.quantise(n, s, o, 1, uvw)
    assert list(q["valid"]) == [1, 1, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0]
    assert (q["i0"][0], q["su"][0], q["i0"][1], q["su"][1]) == (0, 0, 12, 1)
    vis = np.ones((len(uvw), 1), np.complex64)
    g, nv = oracle_mod.grid(n, s, o, 1, 1, uvw, vis, np.ones(len(uvw), np.float32), kernel,
                            return_valid=True)
    assert nv == 2
    assert g.sum() == 2 * s * s
    assert g[7, 0, 0] == 1 and g[7, 15, 0] == 1
    # full-grid footprint S = N = 4: cells 0..3 are those within (-2, 2] of position 1 = centre 2 - 1
    g2 = oracle_mod.grid(4, 4, 1, 1, 1, np.array([[-1, -1, 0]], np.float32), np.ones((1, 1), np.complex64),
                         np.ones(1, np.float32), np.ones((1, 1, 4), np.complex64))
    assert np.all(g2 == 1)


def test_p14_zero_padding_equivalence(oracle_mod):
    # a larger, zero-padded GCF window gives the same grid.  Padding an even
    # number 2c of taps (c each side) moves the footprint origin by -c and keeps the rows.
    n, s, o, c = 40, 6, 4, 2
    uvw, vis, wts, kernel = synth.random_problem(14, 500, n, s, o, 2, 1, spread=0.3)
    g = oracle_mod.grid(n, s, o, 2, 1, uvw, vis, wts, kernel)
    padded = np.zeros((2, o, s + 2 * c), dtype=np.complex64)
    padded[:, :, c:c + s] = kernel
    gp = oracle_mod.grid(n, s + 2 * c, o, 2, 1, uvw, vis, wts, padded)
    assert np.array_equal(g, gp)


def test_p15_thread_count_independence(oracle_mod):
    uvw, vis, wts, kernel = synth.random_problem(15, 5000, 64, 7, 8, 2, 4, spread=0.45, walk=1.5)
    g1 = oracle_mod.grid(64, 7, 8, 2, 4, uvw, vis, wts, kernel, n_threads=1)
    g8 = oracle_mod.grid(64, 7, 8, 2, 4, uvw, vis, wts, kernel, n_threads=8)
    g3 = oracle_mod.grid(64, 7, 8, 2, 4, uvw, vis, wts, kernel, n_threads=3)
    assert np.array_equal(g1, g8) and np.array_equal(g1, g3)
    band = oracle_mod.grid(64, 7, 8, 2, 4, uvw, vis, wts, kernel, rows=(20, 37), n_threads=2)
    assert np.array_equal(band, g1[20:37])


def test_p16_paper_accounting():
    # 365 GGPA/s at 8 flops per grid-point addition is 55 % of 5.288 Tflop/s
    with open(__file__.replace("test_oracle_pins.py", "golden/paper_accounting.txt")) as f:
        vals = dict(line.split("=") for line in f.read().split() if "=" in line)
    eff = float(vals["ggpa_per_s"]) * 1e9 * float(vals["flops_per_gpa"]) / (float(vals["peak_tflops"]) * 1e12)
    assert round(eff * 100) == int(vals["efficiency_percent"])
    assert 7257600 == 2016 * 3600


def test_quantise_matches_independent_python(oracle_mod):
    # Q restated with Python integers / fractions (no float add): rounded oversampled position
    from fractions import Fraction
    import math
    rng = np.random.default_rng(16)
    for (n, s, o) in [(512, 7, 8), (2048, 8, 8), (64, 5, 3), (33, 4, 5)]:
        x = np.concatenate([rng.uniform(-0.6 * n, 0.6 * n, 4000),
                            (rng.integers(-n * o, n * o, 2000) + 0.5) / o]).astype(np.float32)
        uvw = np.zeros((len(x), 3), np.float32)
        uvw[:, 0] = x
        q = oracle_mod.quantise(n, s, o, 1, uvw)
        for k in range(len(x)):
            fx = Fraction(float(x[k]))
            pos = math.floor((fx + n // 2) * o + Fraction(1, 2))        # exact, nearest 1/o, half up
            qi = pos + o - (o * s + 1) // 2
            i0, su = qi // o, qi % o
            ok = 0 <= i0 and i0 + s <= n
            j_ok = q["j0"][k] >= 0
            if ok:
                assert q["valid"][k] == 1 and (q["i0"][k], q["su"][k]) == (i0, su), (n, s, o, x[k])
            else:
                assert q["valid"][k] == 0
            assert j_ok or q["valid"][k] == 0


def test_r4_odd_oversample_times_support_by_hand(oracle_mod):
    """R4 for odd O*S with O > 1, worked on paper for (N, S, O) = (64, 5, 3) (R4 and R8).

    Centre cell 32; the sample is snapped to the nearest 1/3 cell, ties up, and the S = 5 cells of its
    footprint are those at distance d in (-2.5, 2.5] of the snapped position (R8).  Nothing below uses the
    oracle's shift constant O - ceil(O*S/2):
      x = +0.4   -> x*3 = 1.2   -> nearest third 1/3      -> position 32 1/3: cells 30..34 (29 is 3 1/3 away, 35 is 2 2/3) -> i0 = 30
      x =  0.0   ->                nearest third 0        -> position 32    : cells 30..34 (d = -2..2)                    -> i0 = 30
      x = -0.5   -> x*3 = -1.5  -> tie, rounds up to -1/3 -> position 31 2/3: cells 30..34 (29 is 2 2/3 away: outside)     -> i0 = 30
      x = -0.7   -> x*3 = -2.1  -> nearest third -2/3     -> position 31 1/3: cells 29..33 (29 is 2 1/3 away: inside)      -> i0 = 29
      x = +0.9   -> x*3 = 2.7   -> nearest third 1        -> position 33    : cells 31..35                                 -> i0 = 31
    The sub-offset row advances by one per third of a cell and the cell advances when it wraps (R4: q div O, q mod O),
    so the five samples, which sit at thirds -2, -1, 0, +1, +3 of cell 32, must have rows that differ by exactly those
    steps modulo 3 with i0 stepping at the wrap.  The absolute phase of the row for odd O*S (which third is row 0) is
    part of the declared "parity unpinned: physical tap positions" (R8/R24) -- no BASELINE config uses it."""
    xs = np.array([0.4, 0.0, -0.5, -0.7, 0.9], dtype=np.float32)
    uvw = np.zeros((len(xs), 3), np.float32)
    uvw[:, 0] = xs
    q = oracle_mod.quantise(64, 5, 3, 1, uvw)
    assert list(q["valid"]) == [1] * 5
    assert list(q["i0"]) == [30, 30, 30, 29, 31]
    thirds = np.array([1, 0, -1, -2, 3])                       # snapped position in thirds of a cell from cell 32
    lin = np.asarray(q["i0"], dtype=np.int64) * 3 + np.asarray(q["su"], dtype=np.int64)     # q of R4
    assert np.array_equal(lin - lin[1], thirds - thirds[1])   # one row per third, cell carries at the wrap
    assert all(0 <= r < 3 for r in q["su"])
    # the v axis runs through the same code path with the same constants
    uvw2 = np.zeros_like(uvw)
    uvw2[:, 1] = xs
    q2 = oracle_mod.quantise(64, 5, 3, 1, uvw2)
    assert list(q2["j0"]) == [30, 30, 30, 29, 31] and list(q2["sv"]) == list(q["su"])


def test_compress_oracle_runs_and_invariance(oracle_mod):
    # oracle.compress against what its definition fixes: hand-built runs, and the grid of the
    # compressed samples equals the grid of the originals (values chosen exactly representable in float32)
    rng = np.random.default_rng(21)
    base = rng.uniform(-10, 10, (40, 3)).astype(np.float32)
    base[:, 2] = rng.uniform(0, W, 40)
    reps = rng.integers(1, 5, 40)
    uvw = np.repeat(base, reps, axis=0)
    uvw[7] = np.nan                                           # a skipped sample splits / removes a run
    n = len(uvw)
    vis = (rng.integers(-8, 9, (n, 2)) + 1j * rng.integers(-8, 9, (n, 2))).astype(np.complex64)
    wts = rng.integers(1, 4, n).astype(np.float32)
    heads, merged = oracle_mod.compress(N, S, O, W, uvw, vis, wts)
    # expected run heads straight from the construction: one per repeated position, except around the NaN
    starts = np.concatenate([[0], np.cumsum(reps)[:-1]])
    q = oracle_mod.quantise(N, S, O, W, uvw)
    expect = []
    for s0, r in zip(starts, reps):
        idx = [m for m in range(s0, s0 + r) if q["valid"][m]]
        # consecutive valid members form runs; the NaN at 7 may split one
        run = []
        for m in idx:
            if run and m != run[-1] + 1:
                expect.append(run); run = []
            run.append(m)
        if run:
            expect.append(run)
    # neighbouring base positions may coincide after quantisation only by accident; rule that out
    keys = [(q["i0"][r[0]], q["su"][r[0]], q["j0"][r[0]], q["sv"][r[0]], q["wp"][r[0]]) for r in expect]
    assert all(keys[k] != keys[k + 1] or expect[k][-1] + 1 != expect[k + 1][0] for k in range(len(keys) - 1))
    assert list(heads) == [r[0] for r in expect]
    for k, r in enumerate(expect):
        np.testing.assert_array_equal(merged[k], sum(float(wts[m]) * vis[m].astype(np.complex128) for m in r))
    # invariance ("identical results"): merged values are small integers, exact in complex64
    g = oracle_mod.grid(N, S, O, W, 2, uvw, vis, wts, np.ones((W, O, S), np.complex64) * (1 + 0.5j))
    g_c = oracle_mod.grid(N, S, O, W, 2, uvw[heads], merged.astype(np.complex64), np.ones(len(heads), np.float32),
                          np.ones((W, O, S), np.complex64) * (1 + 0.5j))
    np.testing.assert_allclose(g_c, g, rtol=1e-12, atol=1e-12)


def test_dense_oracle_unit_sample_and_separable_limit(oracle_mod):
    # oracle.grid_dense (NEXT-4): (a) one unit visibility reproduces kernel2d[wp][sv][su] with rows = v taps and
    # columns = u taps, at the cell the quantiser gives (hand-placed, asymmetric table so a transpose shows);
    # (b) a dense table that IS an outer product gives exactly the separable oracle's grid
    rng = np.random.default_rng(33)
    k2 = (rng.standard_normal((W, O, O, S, S)) + 1j * rng.standard_normal((W, O, O, S, S))).astype(np.complex64)
    uvw = np.array([[3.0, -4.25, 1.5]], dtype=np.float32)      # Q by hand (N=32, S=5, O=4): su = (12+58) % 4 = 2, sv = (-17+58) % 4 = 1
    q = oracle_mod.quantise(N, S, O, W, uvw)
    assert (q["su"][0], q["sv"][0], q["wp"][0]) == (2, 1, 1)
    g = oracle_mod.grid_dense(N, S, O, W, 1, uvw, np.ones((1, 1), np.complex64), np.ones(1, np.float32), k2)
    expect = np.zeros((N, N), np.complex128)
    expect[q["j0"][0]:q["j0"][0] + S, q["i0"][0]:q["i0"][0] + S] = k2[1, 1, 2].astype(np.complex128)
    np.testing.assert_array_equal(g[:, :, 0], expect)
    uvw, vis, wts, kernel = synth.random_problem(34, 700, N, S, O, W, 2, spread=0.5)
    kk = kernel.astype(np.complex128)
    outer = (kk[:, :, None, :, None] * kk[:, None, :, None, :])        # [wp][sv][su][tj][ti] = k[wp][sv][tj] * k[wp][su][ti]
    g_sep = oracle_mod.grid(N, S, O, W, 2, uvw, vis, wts, kernel)
    # the outer product is not exactly representable in complex64: compare through the rounded table's own error
    g_dense = oracle_mod.grid_dense(N, S, O, W, 2, uvw, vis, wts, outer.astype(np.complex64))
    assert np.abs(g_dense - g_sep).max() <= 4e-7 * np.abs(g_sep).max()
    assert np.linalg.norm(g_dense - g_sep) <= 2e-7 * np.linalg.norm(g_sep)


def test_dense_pol_oracle_unit_sample_per_polarisation_and_equal_limit(oracle_mod):
    # oracle.grid_dense_pol (NEXT-4 remainder), pinned by what its definition fixes:
    # (a) one sample with a DIFFERENT unit visibility per polarisation reproduces, in each polarisation plane of the
    #     grid, that polarisation's own table entry kernel2d[p][wp][sv][su] times that visibility -- rows = v taps,
    #     columns = u taps, at the hand-quantised cell (asymmetric random tables: a swapped polarisation, a transpose
    #     or a wrong sub-offset order shows);
    # (b) with the same table for every polarisation it is exactly oracle.grid_dense (bit for bit: same arithmetic);
    # (c) linearity in the table: scaling polarisation 1's table by 2 doubles plane 1 of the grid and nothing else.
    rng = np.random.default_rng(41)
    P = 4
    k2 = (rng.standard_normal((P, W, O, O, S, S)) + 1j * rng.standard_normal((P, W, O, O, S, S))).astype(np.complex64)
    uvw = np.array([[3.0, -4.25, 1.5]], dtype=np.float32)      # as in the dense pin: su = 2, sv = 1, plane 1 (N=32, S=5, O=4)
    q = oracle_mod.quantise(N, S, O, W, uvw)
    assert (q["su"][0], q["sv"][0], q["wp"][0]) == (2, 1, 1)
    v = np.array([[1.0, 2.0, 1j, -1.0 - 1j]], dtype=np.complex64)
    g = oracle_mod.grid_dense_pol(N, S, O, W, P, uvw, v, np.ones(1, np.float32), k2)
    j0, i0 = q["j0"][0], q["i0"][0]
    for p in range(P):
        expect = np.zeros((N, N), np.complex128)
        expect[j0:j0 + S, i0:i0 + S] = complex(v[0, p]) * k2[p, 1, 1, 2].astype(np.complex128)
        np.testing.assert_array_equal(g[:, :, p], expect)
    uvw, vis, wts, _ = synth.random_problem(42, 500, N, S, O, W, P, spread=0.5)
    same = np.broadcast_to(k2[2], k2.shape).copy()
    np.testing.assert_array_equal(oracle_mod.grid_dense_pol(N, S, O, W, P, uvw, vis, wts, same),
                                  oracle_mod.grid_dense(N, S, O, W, P, uvw, vis, wts, k2[2]))
    g1 = oracle_mod.grid_dense_pol(N, S, O, W, P, uvw, vis, wts, k2)
    k3 = k2.copy()
    k3[1] *= 2
    g2 = oracle_mod.grid_dense_pol(N, S, O, W, P, uvw, vis, wts, k3)
    np.testing.assert_array_equal(g2[:, :, 1], 2 * g1[:, :, 1])
    np.testing.assert_array_equal(g2[:, :, [0, 2, 3]], g1[:, :, [0, 2, 3]])
