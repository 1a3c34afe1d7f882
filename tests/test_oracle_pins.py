"""Pins of the CPU oracle (oracle/cc_oracle.c) against what the paper and the
mathematics fix -- never against itself and never against the CUDA path.

P1  integer circular shifts recovered exactly            (PAPER.md:L55 periodic b.c.)
P2  Parseval                                              (DFT invariant)
P3  direct correlation == DFT correlation                 (Eq. (4))
P4  upsampled values at integer offsets == cc             (ties stage 2 to stage 1)
P5  local upsampled window == zero-padded inverse DFT     ("as if the
    original image had u^2 x the pixels"; textbook trigonometric interpolation)
P6  Fourier-shift theorem, fractional shifts on the 1/u grid recovered exactly
P7  noiseless Gaussian spots recovered to 1e-4 px         (north_star)
P8  self-correlation: d = 0, peak = sum I^2
P9  factored == unfactored upsampled DFT
P10 invariances (constant offsets, positive scaling, integer rolls)
P0  worked size example of the paper: u = 256 -> 384 samples
numpy.fft is used here only as an independent library routine to cross-check
the naive DFT (a "special case that reduces to a library routine").
"""
import numpy as np
import pytest


def _rng(seed):
    return np.random.default_rng(seed)


def _int_image(rng, H, W, hi=200):
    return rng.integers(0, hi, size=(H, W)).astype(np.float64)


def _track_f(oracle, frame, ref, u):
    """Oracle path on float64 images (pins need non-integer inputs too)."""
    cc, P = oracle.cc_dft(frame, ref)
    H, W = cc.shape
    i = oracle.argmax(cc)
    y0, x0 = divmod(i, W)
    wy = y0 - H if 2 * y0 >= H else y0
    wx = x0 - W if 2 * x0 >= W else x0
    up = oracle.upsampled(P, u, y0, x0, want_grid=False)
    M = oracle.grid_size(u)
    c = M // 2
    return dict(wy=wy, wx=wx, m=up["m"], n=up["n"], c=c,
                dy=wy + (up["m"] - c) / u, dx=wx + (up["n"] - c) / u,
                peak=up["top1"], cc=cc, P=P, y0=y0, x0=x0)


# ---------------------------------------------------------------- P0
def test_p0_grid_size_worked_example(oracle_mod):
    # golden: tests/golden/grid_size.txt -- "When u = 256 ... 384 x 384"
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "grid_size.txt")
    rows = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    for u, M in rows:
        assert oracle_mod.grid_size(int(u)) == int(M)


# ---------------------------------------------------------------- DFT vs library / literal
@pytest.mark.parametrize("shape", [(8, 8), (12, 16), (16, 6), (7, 9)])
def test_dft2_matches_literal_and_library(oracle_mod, shape):
    img = _int_image(_rng(1), *shape)
    F = oracle_mod.dft2(img)
    Fl = oracle_mod.dft2(img, literal=True)
    Fn = np.fft.fft2(img)
    s = np.abs(Fn).max()
    assert np.abs(F - Fl).max() <= 1e-12 * s
    assert np.abs(F - Fn).max() <= 1e-12 * s
    back = oracle_mod.idft2(F)
    assert np.abs(back.real - img).max() <= 1e-12 * img.max()
    assert np.abs(back.imag).max() <= 1e-12 * img.max()


def test_dft2_delta_and_plane_wave(oracle_mod):
    # closed forms: delta at (a,b) -> pure phase; cos plane wave -> two bins
    H, W = 8, 16
    img = np.zeros((H, W)); img[3, 5] = 1.0
    F = oracle_mod.dft2(img)
    ky, kx = np.meshgrid(np.arange(H), np.arange(W), indexing="ij")
    assert np.abs(F - np.exp(-2j * np.pi * (ky * 3 / H + kx * 5 / W))).max() < 1e-13
    y, x = np.meshgrid(np.arange(H), np.arange(W), indexing="ij")
    img = np.cos(2 * np.pi * (2 * y / H + 3 * x / W))
    F = oracle_mod.dft2(img)
    exp = np.zeros((H, W), complex); exp[2, 3] = H * W / 2; exp[H - 2, W - 3] = H * W / 2
    assert np.abs(F - exp).max() < 1e-11


# ---------------------------------------------------------------- P2
def test_p2_parseval(oracle_mod):
    rng = _rng(2)
    H, W = 16, 24
    I, E = _int_image(rng, H, W), _int_image(rng, H, W)
    F, G = oracle_mod.dft2(I), oracle_mod.dft2(E)
    assert abs((np.abs(F) ** 2).sum() / (H * W) - (I * I).sum()) <= 1e-12 * (I * I).sum()
    assert abs((np.abs(G) ** 2).sum() / (H * W) - (E * E).sum()) <= 1e-12 * (E * E).sum()
    cc, P = oracle_mod.cc_dft(I, E)
    cross = (I * E).sum()
    assert abs((F * G.conj()).sum().real / (H * W) - cross) <= 1e-12 * cross
    assert abs(cc[0, 0] - cross) <= 1e-12 * cross


# ---------------------------------------------------------------- P3
@pytest.mark.parametrize("shape", [(8, 8), (16, 16), (12, 16), (5, 7)])
def test_p3_direct_equals_dft_correlation(oracle_mod, shape):
    rng = _rng(3)
    I, E = _int_image(rng, *shape), _int_image(rng, *shape)
    cc, _ = oracle_mod.cc_dft(I, E)
    ccd = oracle_mod.cc_direct(I, E)
    assert np.abs(cc - ccd).max() <= 1e-9 * np.abs(ccd).max()
    assert oracle_mod.argmax(cc) == oracle_mod.argmax(ccd)
    # brute force of the brute force, in numpy, on the defining sum of Eq. (4)
    H, W = shape
    s = (2 % H, 3 % W)
    val = sum(I[(y + s[0]) % H, (x + s[1]) % W] * E[y, x] for y in range(H) for x in range(W))
    assert abs(ccd[s] - val) <= 1e-9 * abs(val)


# ---------------------------------------------------------------- P1 / P8
def test_p1_integer_circular_shifts_all_lags_tiny(oracle_mod):
    rng = _rng(4)
    H, W, u = 8, 8, 4
    ref = _int_image(rng, H, W)
    M = oracle_mod.grid_size(u); c = M // 2
    for a in range(H):
        for b in range(W):
            frame = np.roll(ref, (a, b), axis=(0, 1))
            r = _track_f(oracle_mod, frame, ref, u)
            assert (r["wy"], r["wx"]) == (a - H if 2 * a >= H else a, b - W if 2 * b >= W else b)
            assert (r["m"], r["n"]) == (c, c)
            assert abs(r["peak"] - (ref * ref).sum()) <= 1e-12 * (ref * ref).sum()


@pytest.mark.parametrize("H,W,u", [(64, 64, 100), (32, 128, 20), (128, 32, 7)])
def test_p1_integer_circular_shifts_through_track(oracle_mod, H, W, u):
    rng = _rng(5)
    ref_px = rng.integers(0, 4000, size=(H, W)).astype(np.uint16)
    sh = [(0, 0), (1, 0), (0, -1), (H // 2 - 1, W // 2 - 1), (-H // 2, -W // 2), (5, -17 % W)]
    frames = np.stack([np.roll(ref_px, s, axis=(0, 1)) for s in sh])
    r = oracle_mod.track(frames, ref_px.astype(np.float32), u)
    e2 = (ref_px.astype(np.float64) ** 2).sum()
    for i, (a, b) in enumerate(sh):
        a = (a + H // 2) % H - H // 2
        b = (b + W // 2) % W - W // 2
        assert (r.wy[i], r.wx[i]) == (a, b)
        assert r.dy[i] == a and r.dx[i] == b          # sub-pixel offset exactly 0
        assert abs(r.peak[i] - e2) <= 1e-12 * e2      # P8 for shift (0,0): peak = sum I^2
        assert r.cc_top1[i] > r.cc_top2[i]


# ---------------------------------------------------------------- P4
@pytest.mark.parametrize("H,W,u", [(8, 8, 2), (12, 16, 4), (9, 7, 2)])
def test_p4_integer_offsets_reproduce_cc(oracle_mod, H, W, u):
    rng = _rng(6)
    I, E = _int_image(rng, H, W), _int_image(rng, H, W)
    cc, P = oracle_mod.cc_dft(I, E)
    y0, x0 = divmod(oracle_mod.argmax(cc), W)
    up = oracle_mod.upsampled(P, u, y0, x0)
    M = oracle_mod.grid_size(u); c = M // 2
    hits = 0
    for m in range(M):
        for n in range(M):
            if (m - c) % u == 0 and (n - c) % u == 0:
                j, i = (m - c) // u, (n - c) // u
                ref = cc[(y0 + j) % H, (x0 + i) % W]
                assert abs(up["C"][m, n] - ref) <= 1e-12 * np.abs(cc).max()
                hits += 1
    assert hits >= 1


# ---------------------------------------------------------------- P5
def _zero_padded_upsample(P, u):
    """Textbook trigonometric interpolation: embed the H x W spectrum in a
    uH x uW one (Nyquist bins of even axes split half/half), inverse DFT
    (numpy, library routine), scale u^2."""
    H, W = P.shape

    def embed_axis(A, N, axis):
        A = np.moveaxis(A, axis, 0)
        big = np.zeros((u * N,) + A.shape[1:], complex)
        for k in range(N):
            f = k if 2 * k < N else k - N
            if N % 2 == 0 and 2 * k == N:
                big[N // 2] += 0.5 * A[k]
                big[u * N - N // 2] += 0.5 * A[k]
            else:
                big[f % (u * N)] += A[k]
        return np.moveaxis(big, 0, axis)

    big = embed_axis(embed_axis(P, H, 0), W, 1)
    return np.fft.ifft2(big) * (u * u)


@pytest.mark.parametrize("H,W,u", [(8, 8, 2), (12, 16, 4), (8, 8, 4), (7, 10, 2)])
def test_p5_window_of_zero_padded_inverse_dft(oracle_mod, H, W, u):
    rng = _rng(7)
    I, E = _int_image(rng, H, W), _int_image(rng, H, W)
    cc, P = oracle_mod.cc_dft(I, E)
    full = _zero_padded_upsample(P, u)
    assert np.abs(full.imag).max() <= 1e-10 * np.abs(full.real).max()
    y0, x0 = divmod(oracle_mod.argmax(cc), W)
    up = oracle_mod.upsampled(P, u, y0, x0)
    M = oracle_mod.grid_size(u); c = M // 2
    for m in range(M):
        for n in range(M):
            ref = full.real[(y0 * u + m - c) % (u * H), (x0 * u + n - c) % (u * W)]
            assert abs(up["C"][m, n] - ref) <= 1e-12 * np.abs(full.real).max()
    # interp_at (general real lag) agrees with the grid at grid lags
    v = oracle_mod.interp_at(P, y0 + (1 - c) / u, x0 + (2 - c) / u)
    assert abs(v - up["C"][1, 2]) <= 1e-12 * np.abs(full.real).max()


# ---------------------------------------------------------------- P9
@pytest.mark.parametrize("H,W,u", [(8, 8, 3), (6, 10, 4)])
def test_p9_factored_equals_unfactored(oracle_mod, H, W, u):
    rng = _rng(8)
    I, E = _int_image(rng, H, W), _int_image(rng, H, W)
    cc, P = oracle_mod.cc_dft(I, E)
    y0, x0 = divmod(oracle_mod.argmax(cc), W)
    a = oracle_mod.upsampled(P, u, y0, x0)
    b = oracle_mod.upsampled(P, u, y0, x0, literal=True)
    assert np.abs(a["C"] - b["C"]).max() <= 1e-12 * np.abs(b["C"]).max()
    assert (a["m"], a["n"]) == (b["m"], b["n"])
    # argmax bookkeeping of cco_upsampled against numpy on its own grid
    i = int(np.argmax(a["C"]))
    assert (a["m"], a["n"]) == divmod(i, a["C"].shape[1])
    srt = np.sort(a["C"].ravel())
    assert a["top1"] == srt[-1] and a["top2"] == srt[-2]


# ---------------------------------------------------------------- P6
def _fourier_shift(ref, dy, dx):
    """Band-limited ref (Nyquist rows/cols already zero) shifted by (dy, dx)
    through the phase ramp (library FFT; shift theorem)."""
    H, W = ref.shape
    fy = np.fft.fftfreq(H)[:, None]
    fx = np.fft.fftfreq(W)[None, :]
    return np.fft.ifft2(np.fft.fft2(ref) * np.exp(-2j * np.pi * (fy * dy + fx * dx))).real


@pytest.mark.parametrize("u,delta", [(10, (0.3, -0.7)), (10, (2.4, 5.0)), (20, (-3.35, 1.7)),
                                     (4, (0.25, 0.5))])
def test_p6_fourier_shift_theorem(oracle_mod, u, delta):
    rng = _rng(9)
    H, W = 16, 20
    ref = rng.normal(size=(H, W)) + 5.0
    Fr = np.fft.fft2(ref); Fr[H // 2, :] = 0; Fr[:, W // 2] = 0
    ref = np.fft.ifft2(Fr).real
    frame = _fourier_shift(ref, *delta)
    r = _track_f(oracle_mod, frame, ref, u)
    assert abs(r["dy"] - delta[0]) <= 1e-12 and abs(r["dx"] - delta[1]) <= 1e-12
    e2 = (ref * ref).sum()
    assert abs(r["peak"] - e2) <= 1e-11 * e2


# ---------------------------------------------------------------- P7
def _gauss_spot(H, W, cy, cx, sigma, amp=1000.0, bg=10.0):
    y = np.arange(H)[:, None]; x = np.arange(W)[None, :]
    return amp * np.exp(-((y - cy) ** 2 + (x - cx) ** 2) / (2 * sigma ** 2)) + bg


def test_p7_gaussian_on_grid_shifts_exact(oracle_mod):
    H = W = 64; u = 100
    ref = _gauss_spot(H, W, 32, 32, 3.0)
    for sy, sx in [(0.37, -1.42), (-4.99, 3.5), (2.0, 0.01), (-0.74, 0.74)]:
        r = _track_f(oracle_mod, _gauss_spot(H, W, 32 + sy, 32 + sx, 3.0), ref, u)
        assert abs(r["dy"] - sy) < 1e-9 and abs(r["dx"] - sx) < 1e-9


def test_p7_gaussian_arbitrary_shifts_to_1e_4(oracle_mod):
    # u = 5000 -> grid spacing 2e-4, so the nearest grid point is within 1e-4 px
    H = W = 32; u = 5000
    ref = _gauss_spot(H, W, 16, 16, 2.5)
    for sy, sx in [(1.234567, -2.718281), (-3.141592, 0.577215)]:
        r = _track_f(oracle_mod, _gauss_spot(H, W, 16 + sy, 16 + sx, 2.5), ref, u)
        assert abs(r["dy"] - sy) <= 1e-4 + 1e-9 and abs(r["dx"] - sx) <= 1e-4 + 1e-9


# ---------------------------------------------------------------- P10 + degenerate cases
def test_p10_invariances(oracle_mod):
    rng = _rng(10)
    H, W, u = 16, 16, 8
    ref = _gauss_spot(H, W, 8, 8, 1.7, amp=300, bg=4) + rng.normal(size=(H, W))
    frame = _gauss_spot(H, W, 9.3, 6.6, 1.7, amp=300, bg=4) + rng.normal(size=(H, W))
    base = _track_f(oracle_mod, frame, ref, u)
    r = _track_f(oracle_mod, frame + 37.0, ref, u)
    assert (r["dy"], r["dx"]) == (base["dy"], base["dx"])
    r = _track_f(oracle_mod, frame, ref + 11.0, u)
    assert (r["dy"], r["dx"]) == (base["dy"], base["dx"])
    r = _track_f(oracle_mod, 3.0 * frame, 0.5 * ref, u)
    assert (r["dy"], r["dx"]) == (base["dy"], base["dx"])
    assert abs(r["peak"] - 1.5 * base["peak"]) <= 1e-12 * abs(base["peak"])
    r = _track_f(oracle_mod, np.roll(frame, (2, -3), axis=(0, 1)), ref, u)
    assert abs(r["dy"] - (base["dy"] + 2)) < 1e-12 and abs(r["dx"] - (base["dx"] - 3)) < 1e-12


def test_constant_frame_degenerate_case(oracle_mod):
    # cc constant -> (y0,x0) = (0,0); C constant up to rounding is NOT guaranteed
    # in floating point, so use frame = 0: everything is exactly 0 and the
    # smallest-index rule decides: (m*,n*) = (0,0), d = (-c/u, -c/u).
    H, W, u = 8, 8, 4
    frames = np.zeros((1, H, W), np.uint8)
    ref = _rng(11).random((H, W)).astype(np.float32)
    r = oracle_mod.track(frames, ref, u)
    c = oracle_mod.grid_size(u) // 2
    assert (r.wy[0], r.wx[0], r.m[0], r.n[0]) == (0, 0, 0, 0)
    assert r.dy[0] == -c / u and r.dx[0] == -c / u and r.peak[0] == 0.0


def test_exact_tie_smallest_index(oracle_mod):
    # reference = single bright pixel, frame = two equal bright pixels:
    # cc has two exactly equal maxima (integers, exact in double); the smaller
    # row-major index must win.
    H, W = 8, 8
    ref = np.zeros((H, W), np.float32); ref[0, 0] = 2.0
    fr = np.zeros((1, H, W), np.uint16); fr[0, 1, 5] = 7; fr[0, 3, 2] = 7
    r = oracle_mod.track(fr, ref, 1)
    assert (r.wy[0], r.wx[0]) == (1, 5 - W)
    assert r.cc_top1[0] == r.cc_top2[0] == 14.0


def test_upsample_one_is_integer_peak_only(oracle_mod):
    rng = _rng(12)
    fr = rng.integers(0, 255, size=(3, 8, 16)).astype(np.uint8)
    ref = rng.random((8, 16)).astype(np.float32)
    r = oracle_mod.track(fr, ref, 1)
    for i in range(3):
        cc = oracle_mod.cc_direct(fr[i].astype(float), ref.astype(float))
        y0, x0 = divmod(int(np.argmax(cc)), 16)
        assert (r.wy[i], r.wx[i]) == (y0 - 8 if y0 >= 4 else y0, x0 - 16 if x0 >= 8 else x0)
        assert r.dy[i] == r.wy[i] and r.dx[i] == r.wx[i]


def test_track_matches_piecewise_pipeline(oracle_mod):
    # cco_track (pixels in, result out) equals the step-by-step calls
    from paper_2310_08770_b200 import workloads as wl
    cfg = wl.config(1)
    fr = wl.frames(cfg, [3, 7]); ref = wl.reference(cfg)
    r = oracle_mod.track(fr, ref, cfg.upsample)
    for i in range(2):
        p = _track_f(oracle_mod, fr[i].astype(np.float64), ref.astype(np.float64), cfg.upsample)
        assert (p["wy"], p["wx"], p["m"], p["n"]) == (r.wy[i], r.wx[i], r.m[i], r.n[i])
        assert p["dy"] == r.dy[i] and p["dx"] == r.dx[i]


def test_p11_shot_noise_sanity_band(oracle_mod):
    # informational band: CC-U error within ~1x-3x of the
    # shot-noise limit w0/(2 sqrt(N_gamma)) = sigma/sqrt(N_gamma)
    from paper_2310_08770_b200 import workloads as wl
    cfg = wl.config(1)
    idx = np.arange(48)
    r = oracle_mod.track(wl.frames(cfg, idx), wl.reference(cfg), cfg.upsample)
    s = wl.shifts(cfg)[idx]
    err = np.sqrt(np.mean((r.dy - s[:, 0]) ** 2 + (r.dx - s[:, 1]) ** 2) / 2)
    limit = 3.0 / np.sqrt(2 * np.pi * 9 * 1000)
    assert 0.5 * limit < err < 4.0 * limit


# ---------------------------------------------------------------- CC-SN (Eqs. (5)-(7))
# SN1  Cauchy-Schwarz closed form: frame = circshift(ref) -> d = shift, minimum value = sum(E + eps)
# SN2  brute-force left-hand side of Eq. (7) on tiny frames: same integer minimiser, same minimum
# SN3  chi^2 of Eq. (6) itself (all three terms) is minimised at the oracle's integer peak
# SN4  large eps -> CC-SN results approach CC-U
# SN5  common positive scaling of (I', E') leaves d unchanged; value scales linearly

def _sn_direct(I, E, eps):
    """S(s) = sum_r (I(r+s) + eps)^2 / (E(r) + eps), literal double loop over lags (Eq. (7), left side)."""
    H, W = I.shape
    Ip2 = (I + eps) ** 2
    w = 1.0 / (E + eps)
    S = np.empty((H, W))
    for sy in range(H):
        for sx in range(W):
            S[sy, sx] = np.sum(np.roll(Ip2, (-sy, -sx), axis=(0, 1)) * w)
    return S


@pytest.mark.parametrize("H,W,u,eps", [(16, 16, 4, 7.5), (32, 64, 10, 0.0), (64, 64, 20, 200.0)])
def test_sn1_circular_shift_closed_form(oracle_mod, H, W, u, eps):
    rng = _rng(21)
    ref = rng.integers(3, 900, size=(H, W)).astype(np.float32)
    shifts = [(0, 0), (1, 0), (0, 1), (H // 2, W // 2), (H - 1, W - 1), (5, W - 7)]
    fr = np.stack([np.roll(ref, s, axis=(0, 1)) for s in shifts]).astype(np.uint16)
    o = oracle_mod.track(fr, ref, u, method="sn", epsilon=eps)
    for k, (a, b) in enumerate(shifts):
        wa = a - H if 2 * a >= H else a
        wb = b - W if 2 * b >= W else b
        assert (o.wy[k], o.wx[k]) == (wa, wb)
        assert o.dy[k] == wa and o.dx[k] == wb           # (sum I')^2 <= S * sum E' with equality iff aligned
    assert np.allclose(o.peak, np.sum(ref.astype(np.float64) + eps), rtol=1e-12)


@pytest.mark.parametrize("shape,eps", [((8, 8), 3.0), ((12, 16), 50.0)])
def test_sn2_brute_force_eq7(oracle_mod, shape, eps):
    rng = _rng(22)
    H, W = shape
    ref = rng.integers(1, 300, size=shape).astype(np.float32)
    fr = rng.integers(0, 300, size=(5,) + shape).astype(np.uint8)
    o = oracle_mod.track(fr, ref, 1, method="sn", epsilon=eps)
    for k in range(5):
        S = _sn_direct(fr[k].astype(np.float64), ref.astype(np.float64), eps)
        i = int(np.argmin(S))                              # first index among equal minima
        y0, x0 = divmod(i, W)
        assert (o.wy[k], o.wx[k]) == (y0 - H if 2 * y0 >= H else y0, x0 - W if 2 * x0 >= W else x0)
        assert abs(o.peak[k] / S.min() - 1) < 1e-12
        assert abs(o.cc_top2[k] / np.partition(S.ravel(), 1)[1] - 1) < 1e-12


def test_sn3_minimises_chi2_of_eq6(oracle_mod):
    """chi^2(s) = sum_r { E' - 2 I'(r+s) + I'(r+s)^2 / E' }: the oracle's integer peak is its minimiser."""
    rng = _rng(23)
    H, W, eps = 12, 12, 4.0
    y, x = np.mgrid[0:H, 0:W]
    ref = (100.0 * np.exp(-((y - 6) ** 2 + (x - 6) ** 2) / 6.0) + 5.0).astype(np.float32)
    fr = rng.poisson(np.roll(ref.astype(np.float64), (2, -3), axis=(0, 1))).astype(np.uint16)[None]
    o = oracle_mod.track(fr, ref, 1, method="sn", epsilon=eps)
    Ep, Ip = ref.astype(np.float64) + eps, fr[0].astype(np.float64) + eps
    chi2 = np.array([[np.sum(Ep - 2 * np.roll(Ip, (-sy, -sx), axis=(0, 1)) + np.roll(Ip, (-sy, -sx), axis=(0, 1)) ** 2 / Ep)
                      for sx in range(W)] for sy in range(H)])
    y0, x0 = divmod(int(np.argmin(chi2)), W)
    assert (o.wy[0] % H, o.wx[0] % W) == (y0, x0) == (2, W - 3)


def test_sn4_large_offset_approaches_ccu(oracle_mod):
    """"for larger values [of eps] the CC-SN method's results approach those of the CC-U method"."""
    from paper_2310_08770_b200 import workloads as wl
    cfg = wl.config(1)
    fr = wl.frames(cfg, np.arange(24))
    ref = wl.reference(cfg)
    ou = oracle_mod.track(fr, ref, 20)
    far = oracle_mod.track(fr, ref, 20, method="sn", epsilon=1e7)
    near = oracle_mod.track(fr, ref, 20, method="sn", epsilon=1.0)
    d_far = np.hypot(far.dx - ou.dx, far.dy - ou.dy)
    d_near = np.hypot(near.dx - ou.dx, near.dy - ou.dy)
    assert d_far.max() <= 0.05 + 1e-12 and np.mean(d_far == 0) >= 0.75    # at most one grid step away, mostly identical
    assert d_near.mean() > d_far.mean()                                   # a small offset is a different estimator
    truth = wl.shifts(cfg)[:24]
    assert np.median(np.hypot(near.dx - truth[:, 1], near.dy - truth[:, 0])) < 0.2   # and still tracks the spot


def test_sn5_scaling_invariance(oracle_mod):
    rng = _rng(25)
    ref = rng.integers(10, 120, size=(32, 32)).astype(np.float32)
    fr = np.clip(rng.poisson(np.roll(ref.astype(np.float64), (3, 5), axis=(0, 1)), size=(4, 32, 32)), 0, 120).astype(np.uint16)
    a = oracle_mod.track(fr, ref, 10, method="sn", epsilon=6.0)
    b = oracle_mod.track((2 * fr).astype(np.uint16), 2 * ref, 10, method="sn", epsilon=12.0)   # I', E' both doubled
    assert np.array_equal(a.dx, b.dx) and np.array_equal(a.dy, b.dy)
    assert np.allclose(b.peak, 2 * a.peak, rtol=1e-12)


# ---------------------------------------------------------------- drift correction (Eqs. (10)-(12))
def test_d1_plain_filter_closed_forms(oracle_mod):
    """Eq. (10) with R_0 = a0 r_0: a constant input c gives R_n = c (1 - b1^(n+1)); an impulse gives a0 b1^n."""
    a0, n = 0.05, 200
    c = np.float32(1.25)
    ox, oy, st = oracle_mod.drift_correct(np.full(n, c), np.full(n, -2 * c), a0)
    k = np.arange(1, n + 1)
    assert np.allclose(ox, float(c) * (1 - a0) ** k, rtol=1e-12) and np.allclose(oy, -2 * float(c) * (1 - a0) ** k, rtol=1e-12)
    assert np.allclose(st, [float(c) * (1 - (1 - a0) ** n), -2 * float(c) * (1 - (1 - a0) ** n)], rtol=1e-12)
    imp = np.zeros(50, np.float32)
    imp[0] = 1.0
    ox, _, _ = oracle_mod.drift_correct(imp, imp, 0.2)
    assert np.allclose(ox[1:], -0.2 * 0.8 ** np.arange(1, 50), rtol=1e-12) and abs(ox[0] - 0.8) < 1e-15


def test_d2_rate_limited_steps_exactly_max_step(oracle_mod):
    """Eq. (12): while |dR_n| > alpha/u the offset moves exactly alpha/u along dR_n; afterwards it follows Eq. (10)."""
    a0, step, n = 0.5, 0.005, 40
    rx, ry = np.full(n, 3.0, np.float32), np.full(n, 4.0, np.float32)         # direction (0.6, 0.8), |a0 r| = 2.5 >> step
    ox, oy, st = oracle_mod.drift_correct(rx, ry, a0, step)
    k = np.arange(1, n + 1)
    assert np.allclose(3.0 - ox, 0.6 * step * k, rtol=1e-12) and np.allclose(4.0 - oy, 0.8 * step * k, rtol=1e-12)
    # small input: never clamped -> identical to the plain filter
    rng = np.random.default_rng(3)
    sx, sy = (1e-3 * rng.standard_normal(100)).astype(np.float32), (1e-3 * rng.standard_normal(100)).astype(np.float32)
    a = oracle_mod.drift_correct(sx, sy, 0.1, 0.005)
    b = oracle_mod.drift_correct(sx, sy, 0.1, 0.0)
    assert np.allclose(a[0], b[0], atol=1e-15) and np.allclose(a[1], b[1], atol=1e-15)


def test_d3_state_carries_across_calls_and_linearity(oracle_mod):
    rng = np.random.default_rng(4)
    x, y = rng.standard_normal(300).astype(np.float32), rng.standard_normal(300).astype(np.float32)
    for step in (0.0, 0.005):
        full = oracle_mod.drift_correct(x, y, 0.02, step)
        h1 = oracle_mod.drift_correct(x[:120], y[:120], 0.02, step)
        h2 = oracle_mod.drift_correct(x[120:], y[120:], 0.02, step, state=h1[2])
        assert np.array_equal(np.concatenate([h1[0], h2[0]]), full[0]) and np.array_equal(h2[2], full[2])
    p = oracle_mod.drift_correct(2 * x, 2 * y, 0.02)[0]                       # plain filter is linear
    assert np.allclose(p, 2 * oracle_mod.drift_correct(x, y, 0.02)[0], rtol=1e-12, atol=1e-15)


# ---------------------------------------------------------------- real-time RI update (Eq. (9))
def test_ri1_a0_zero_is_the_fixed_reference(oracle_mod):
    from paper_2310_08770_b200 import workloads as wl
    cfg = wl.config(1)
    fr, ref = wl.frames(cfg, np.arange(6)), wl.reference(cfg)
    a = oracle_mod.track(fr, ref, 20)
    b, G = oracle_mod.track_rt(fr, ref, 20, 0.0)
    assert np.array_equal(a.dx, b.dx) and np.array_equal(a.dy, b.dy) and np.array_equal(a.peak, b.peak)
    assert np.allclose(G, np.fft.fft2(ref.astype(np.float64)), rtol=1e-10, atol=1e-6)


def test_ri2_aligned_copies_leave_the_reference_unchanged(oracle_mod):
    """Frames that are exact translations of the RI (integer circular shifts; fractional shifts of a band-limited
    image by the phase ramp) are shifted back onto it: E_i = a0 E + b1 E = E for every a0.  Fails if the sign of the
    alignment, the Nyquist rule or the filter weights are wrong."""
    rng = _rng(41)
    H, W = 16, 24
    ref = rng.integers(0, 200, size=(H, W)).astype(np.float32)
    shifts = [(3, -5), (0, 7), (-6, 0), (8, 12), (1, 1)]
    fr = np.stack([np.roll(ref, s, axis=(0, 1)) for s in shifts]).astype(np.uint16)
    res, G = oracle_mod.track_rt(fr, ref, 4, 0.3)
    G0 = np.fft.fft2(ref.astype(np.float64))
    assert np.max(np.abs(G - G0)) < 1e-9 * np.max(np.abs(G0))
    for k, (a, b) in enumerate(shifts):
        assert (res.dy[k], res.dx[k]) == (a - H if 2 * a >= H else a, b - W if 2 * b >= W else b)
    # fractional: band-limited reference (Nyquist row/column removed), frames = phase-ramp shifts on the 1/u grid
    u = 8
    B0 = np.fft.fft2(rng.standard_normal((H, W)))
    B0[H // 2, :] = 0
    B0[:, W // 2] = 0
    base = np.real(np.fft.ifft2(B0))
    fy, fx = np.fft.fftfreq(H)[:, None], np.fft.fftfreq(W)[None, :]
    scale = 2000.0 / np.abs(base).max()
    ref2 = np.round(base * scale) + 3000.0                                # integer pixels: quantisation breaks exact
    frames2 = []                                                           # band-limitedness by ~1e-4 relative
    for dy, dx in [(0.375, -0.25), (-1.5, 2.125)]:
        sh = np.real(np.fft.ifft2(np.fft.fft2(ref2) * np.exp(-2j * np.pi * (fy * dy + fx * dx))))
        frames2.append(np.round(sh))
    fr2 = np.stack(frames2).astype(np.uint16)
    res2, G2 = oracle_mod.track_rt(fr2, ref2.astype(np.float32), u, 0.5)
    assert np.allclose(res2.dy, [0.375, -1.5]) and np.allclose(res2.dx, [-0.25, 2.125])
    Gr = np.fft.fft2(ref2)
    err = np.max(np.abs(G2 - Gr))                                          # only the +-0.5 rounding of the pixels remains:
    assert err < 5 * np.sqrt(H * W / 12.0) and err < 1e-2 * np.median(np.abs(Gr))   # ~sqrt(HW/12) per bin, << |G|


def test_ri3_filter_weights_closed_form(oracle_mod):
    """Frames with zero displacement (the RI plus zero-mean noise): no alignment phase, so
    G_n = b1^(n+1) G_ref + a0 sum_k b1^(n-k) F[I_k] -- the low-pass filter of Eq. (9) written out."""
    rng = _rng(42)
    H = W = 16
    y, x = np.mgrid[0:H, 0:W]
    ref = (500.0 * np.exp(-((y - 8) ** 2 + (x - 8) ** 2) / 8.0) + 20.0).astype(np.float32)
    fr = np.clip(np.round(ref[None] + rng.normal(0, 1.0, size=(5, H, W))), 0, 65535).astype(np.uint16)
    a0 = 0.25
    res, G = oracle_mod.track_rt(fr, ref, 2, a0)
    assert np.all(res.dx == 0) and np.all(res.dy == 0)
    expect = (1 - a0) ** 5 * np.fft.fft2(ref.astype(np.float64))
    for k in range(5):
        expect = expect + a0 * (1 - a0) ** (4 - k) * np.fft.fft2(fr[k].astype(np.float64))
    assert np.max(np.abs(G - expect)) < 1e-9 * np.max(np.abs(expect))


# ---------------------------------------------------------------- offline iterative RI (Eq. (8))
def test_it1_mean_of_aligned_images(oracle_mod):
    """Frames = integer circular shifts of one image plus independent noise: after one pass the RI is the plain mean
    of the frames rolled back by their shifts (np.roll + np.mean, no Fourier arithmetic); a second pass keeps d."""
    rng = _rng(61)
    H, W, N = 16, 16, 12
    y, x = np.mgrid[0:H, 0:W]
    base = 400.0 * np.exp(-((y - 8) ** 2 + (x - 8) ** 2) / 6.0) + 30.0
    shifts = rng.integers(-3, 4, size=(N, 2))
    shifts[0] = 0                                                     # E_0 = I_0
    fr = np.stack([np.roll(rng.poisson(base), tuple(s), axis=(0, 1)) for s in shifts]).astype(np.uint16)
    res, G = oracle_mod.iterate_reference(fr, fr[0].astype(np.float32), 1, 1)
    assert np.array_equal(res.wy, shifts[:, 0]) and np.array_equal(res.wx, shifts[:, 1])
    mean = np.mean([np.roll(f.astype(np.float64), tuple(-s), axis=(0, 1)) for f, s in zip(fr, shifts)], axis=0)
    assert np.max(np.abs(G - np.fft.fft2(mean))) < 1e-9 * np.abs(G[0, 0])
    res2, G2 = oracle_mod.iterate_reference(fr, fr[0].astype(np.float32), 1, 2)
    assert np.array_equal(res2.wy, shifts[:, 0]) and np.max(np.abs(G2 - G)) < 1e-9 * np.abs(G[0, 0])


def test_it2_iterations_sharpen_the_reference(oracle_mod):
    """The point of Eq. (8): starting from one noisy frame, the averaged RI approaches the noiseless spot, and the
    rms error of the displacements does not get worse from the first pass to the third."""
    from paper_2310_08770_b200 import workloads as wl
    cfg = wl.config(1)
    fr = wl.frames(cfg, np.arange(40))
    truth = wl.shifts(cfg)[:40]
    clean = wl.reference(cfg).astype(np.float64)
    r1, G1 = oracle_mod.iterate_reference(fr, fr[0].astype(np.float32), 10, 1)
    r3, G3 = oracle_mod.iterate_reference(fr, fr[0].astype(np.float32), 10, 3)
    rel = lambda r: np.hypot((r.dx - r.dx[0]) - (truth[:, 1] - truth[0, 1]), (r.dy - r.dy[0]) - (truth[:, 0] - truth[0, 0]))
    assert np.sqrt(np.mean(rel(r3) ** 2)) <= np.sqrt(np.mean(rel(r1) ** 2)) + 1e-12
    # the averaged RI sits at frame 0's position: compare its spectrum modulus with the clean template's
    noisy = np.abs(np.fft.fft2(fr[0].astype(np.float64)))
    assert np.sum((np.abs(G3) - np.abs(np.fft.fft2(clean))) ** 2) < 0.2 * np.sum((noisy - np.abs(np.fft.fft2(clean))) ** 2)


def test_it3_fractional_alignment_through_the_iteration(oracle_mod):
    """The IT analogue of RI2: frames that are phase-ramp shifts (on the 1/u grid, even H and W) of a band-limited
    image are shifted back onto it by Eq. (8)'s alignment, so after one pass G equals fft2(ref) up to the +-0.5
    rounding of the integer pixels.  Fractional phases and the Nyquist cos(pi d) branch are decisive here: a wrong
    alignment sign doubles the shift instead of removing it (error ~ |G|, five orders above the bound)."""
    rng = _rng(63)
    H, W, u = 16, 24, 8
    B0 = np.fft.fft2(rng.standard_normal((H, W)))
    B0[H // 2, :] = 0
    B0[:, W // 2] = 0
    base = np.real(np.fft.ifft2(B0))
    fy, fx = np.fft.fftfreq(H)[:, None], np.fft.fftfreq(W)[None, :]
    ref = np.round(base * (2000.0 / np.abs(base).max())) + 3000.0
    shifts = [(0.375, -0.25), (-1.5, 2.125), (0.0, 0.0), (2.625, 0.5), (-0.125, -3.75)]
    fr = np.stack([np.round(np.real(np.fft.ifft2(np.fft.fft2(ref) * np.exp(-2j * np.pi * (fy * dy + fx * dx)))))
                   for dy, dx in shifts]).astype(np.uint16)
    res, G = oracle_mod.iterate_reference(fr, ref.astype(np.float32), u, 1)
    assert np.allclose(res.dy, [s[0] for s in shifts]) and np.allclose(res.dx, [s[1] for s in shifts])
    Gr = np.fft.fft2(ref)
    err = np.max(np.abs(G - Gr))
    assert err < 5 * np.sqrt(H * W / 12.0) and err < 1e-2 * np.median(np.abs(Gr))
    # the mean of Eq. (8) is a plain mean: the result does not depend on the order of the frames
    res_p, G_p = oracle_mod.iterate_reference(fr[::-1].copy(), ref.astype(np.float32), u, 1)
    assert np.max(np.abs(G_p - G)) < 1e-9 * np.abs(G[0, 0]) and np.allclose(res_p.dy[::-1], res.dy)


def test_st1_step_from_a_given_spectrum(oracle_mod):
    """cco_step_from_spectrum (the entry the GPU open-loop tests drive): from G = fft2(ref) (library FFT) it returns
    cco_track's displacement; with a0 = 1 the returned spectrum is that of the frame rolled back by its integer shift
    (np.roll, no Fourier arithmetic); with a0 in between, the blend of Eq. (9); a0 = 0 leaves G untouched."""
    rng = _rng(64)
    H, W = 12, 16
    ref = rng.integers(0, 300, size=(H, W)).astype(np.float32)
    G0 = np.fft.fft2(ref.astype(np.float64))
    for (a, b) in [(2, -3), (0, 0), (-5, 7)]:
        frame = np.roll(ref, (a, b), axis=(0, 1)).astype(np.uint16)
        t = oracle_mod.track(frame[None], ref, 4)
        for a0 in (1.0, 0.25, 0.0):
            r, Gn = oracle_mod.step_from_spectrum(frame, G0, 4, a0)
            assert (r.dy[0], r.dx[0]) == (t.dy[0], t.dx[0]) == (float(a), float(b))
            back = np.fft.fft2(np.roll(frame.astype(np.float64), (-a, -b), axis=(0, 1)))
            assert np.max(np.abs(Gn - (a0 * back + (1 - a0) * G0))) < 1e-9 * np.abs(G0[0, 0])
    # a noisy frame against a spectrum that is NOT that of an integer image: same result as the piecewise pipeline
    frame = rng.poisson(ref.astype(np.float64) + 5).astype(np.uint16)
    Gq = G0 * (1.0 + 0.01 * rng.standard_normal(G0.shape))
    Gq = np.fft.fft2(np.real(np.fft.ifft2(Gq)))                          # spectrum of a real image
    r, _ = oracle_mod.step_from_spectrum(frame, Gq, 4, 0.5)
    t = _track_f(oracle_mod, frame.astype(np.float64), np.real(np.fft.ifft2(Gq)), 4)
    assert (r.dy[0], r.dx[0]) == (t["dy"], t["dx"]) and abs(r.peak[0] - t["peak"]) <= 1e-9 * abs(t["peak"])


# ---------------------------------------------------------------- CC-SN with a moving reference image (R19)
# SR1  a0 = 0 is cco_track_sn with the fixed reference
# SR2  exact translations of the RI leave it unchanged; d = shift; S_min = sum(E + eps) (Cauchy-Schwarz, as SN1)
# SR3  eps -> infinity reproduces the CC-U loop of Eq. (9)
# SR4  zero-displacement frames: the state is the low-pass filter of Eq. (9) written out (as RI3)
# SR5  frame i is weighted by 1/(E_{i-1} + eps) with E_{i-1} the UPDATED image average: brute-force Eq. (7)
# SR6  Eq. (8): after one pass the state is the plain mean of the rolled-back frames, and the second pass weights
#      with 1/(that mean + eps): brute-force Eq. (7)
def test_sr1_a0_zero_is_the_fixed_reference(oracle_mod):
    from paper_2310_08770_b200 import workloads as wl
    cfg = wl.config(1)
    fr, ref = wl.frames(cfg, np.arange(6)), wl.reference(cfg)
    a = oracle_mod.track(fr, ref, 20, method="sn", epsilon=50.0)
    b, G = oracle_mod.track_rt(fr, ref, 20, 0.0, method="sn", epsilon=50.0)
    assert np.array_equal(a.dx, b.dx) and np.array_equal(a.dy, b.dy) and np.allclose(a.peak, b.peak, rtol=1e-10)
    assert np.allclose(G, np.fft.fft2(ref.astype(np.float64)), rtol=1e-10, atol=1e-6)


def test_sr2_aligned_copies_leave_the_reference_unchanged(oracle_mod):
    rng = _rng(71)
    H, W, eps = 16, 24, 12.5
    ref = rng.integers(3, 200, size=(H, W)).astype(np.float32)
    shifts = [(3, -5), (0, 7), (-6, 0), (8, 12), (1, 1)]
    fr = np.stack([np.roll(ref, s, axis=(0, 1)) for s in shifts]).astype(np.uint16)
    G0 = np.fft.fft2(ref.astype(np.float64))
    for a0 in (0.3, 1.0):
        res, G = oracle_mod.track_rt(fr, ref, 4, a0, method="sn", epsilon=eps)
        assert np.max(np.abs(G - G0)) < 1e-9 * np.max(np.abs(G0))
        for k, (a, b) in enumerate(shifts):
            assert (res.dy[k], res.dx[k]) == (a - H if 2 * a >= H else a, b - W if 2 * b >= W else b)
        assert np.allclose(res.peak, np.sum(ref.astype(np.float64) + eps), rtol=1e-10)
    res, G = oracle_mod.iterate_reference(fr, ref, 4, 2, method="sn", epsilon=eps)
    assert np.max(np.abs(G - G0)) < 1e-9 * np.max(np.abs(G0)) and np.allclose(res.peak, np.sum(ref.astype(np.float64) + eps), rtol=1e-10)


def test_sr3_large_offset_reproduces_the_ccu_loop(oracle_mod):
    """PAPER.md:L161 for the closed loop: with eps = 1e7 the weights are flat, the displacements are those of the CC-U
    loop (at most one grid step away, mostly identical) and so is the running reference."""
    from paper_2310_08770_b200 import workloads as wl
    cfg = wl.config(1)
    fr, ref = wl.frames(cfg, np.arange(16)), wl.reference(cfg)
    ru, Gu = oracle_mod.track_rt(fr, ref, 20, 0.2)
    rs, Gs = oracle_mod.track_rt(fr, ref, 20, 0.2, method="sn", epsilon=1e7)
    d = np.hypot(rs.dx - ru.dx, rs.dy - ru.dy)
    assert d.max() <= 0.05 * np.sqrt(2) + 1e-12 and np.mean(d == 0) >= 0.75
    scale = np.max(np.abs(Gu[1:, 1:]))
    assert np.max(np.abs(Gs - Gu)) < 2e-2 * scale
    near, _ = oracle_mod.track_rt(fr, ref, 20, 0.2, method="sn", epsilon=1.0)
    assert np.hypot(near.dx - ru.dx, near.dy - ru.dy).mean() > d.mean()       # a small offset is a different estimator


def test_sr4_filter_weights_closed_form(oracle_mod):
    rng = _rng(72)
    H = W = 16
    y, x = np.mgrid[0:H, 0:W]
    ref = (500.0 * np.exp(-((y - 8) ** 2 + (x - 8) ** 2) / 8.0) + 20.0).astype(np.float32)
    fr = np.clip(np.round(ref[None] + rng.normal(0, 1.0, size=(5, H, W))), 0, 65535).astype(np.uint16)
    a0 = 0.25
    res, G = oracle_mod.track_rt(fr, ref, 2, a0, method="sn", epsilon=30.0)
    assert np.all(res.dx == 0) and np.all(res.dy == 0)
    expect = (1 - a0) ** 5 * np.fft.fft2(ref.astype(np.float64))
    for k in range(5):
        expect = expect + a0 * (1 - a0) ** (4 - k) * np.fft.fft2(fr[k].astype(np.float64))
    assert np.max(np.abs(G - expect)) < 1e-9 * np.max(np.abs(expect))


def test_sr5_weight_follows_the_updated_reference(oracle_mod):
    """Frame 0 sits on the RI (d_0 = 0), so E_0 = a0 I_0 + b1 E_{-1} pixel by pixel (no Fourier arithmetic); frame 1
    must then be measured with the weight 1/(E_0 + eps): integer minimiser, minimum and runner-up of the literal
    double loop of Eq. (7).  Fails for a stale weight 1/(E_{-1} + eps) and for the literal substitution of L92."""
    rng = _rng(73)
    H, W, eps, a0 = 10, 12, 6.0, 0.6
    y, x = np.mgrid[0:H, 0:W]
    ref = (150.0 * np.exp(-((y - 5) ** 2 + (x - 6) ** 2) / 5.0) + 8.0).astype(np.float32)
    f0 = rng.poisson(ref.astype(np.float64)).astype(np.uint16)
    f1 = rng.poisson(np.roll(ref.astype(np.float64), (2, -3), axis=(0, 1))).astype(np.uint16)
    res, G = oracle_mod.track_rt(np.stack([f0, f1]), ref, 1, a0, method="sn", epsilon=eps)
    assert (res.dy[0], res.dx[0]) == (0.0, 0.0)
    E0 = a0 * f0.astype(np.float64) + (1 - a0) * ref.astype(np.float64)
    S = _sn_direct(f1.astype(np.float64), E0, eps)
    y0, x0 = divmod(int(np.argmin(S)), W)
    assert (res.wy[1] % H, res.wx[1] % W) == (y0, x0) == (2, W - 3)
    assert abs(res.peak[1] / S.min() - 1) < 1e-11 and abs(res.cc_top2[1] / np.partition(S.ravel(), 1)[1] - 1) < 1e-11
    stale = _sn_direct(f1.astype(np.float64), ref.astype(np.float64), eps)
    assert abs(res.peak[1] / stale.min() - 1) > 1e-4                          # the pin can tell the two apart
    # one step from a given state gives the same answer (cco_step_from_spectrum_sn)
    r1, _ = oracle_mod.step_from_spectrum(f1, np.fft.fft2(E0), 1, a0, method="sn", epsilon=eps)
    assert (r1.dy[0], r1.dx[0]) == (res.dy[1], res.dx[1]) and abs(r1.peak[0] / res.peak[1] - 1) < 1e-11
    with pytest.raises(ValueError):                                           # E + eps must stay positive
        oracle_mod.step_from_spectrum(f1, np.fft.fft2(E0 - 200.0), 1, a0, method="sn", epsilon=eps)


def test_sr6_offline_passes(oracle_mod):
    rng = _rng(74)
    H, W, N, eps = 12, 12, 10, 9.0
    y, x = np.mgrid[0:H, 0:W]
    base = 400.0 * np.exp(-((y - 6) ** 2 + (x - 6) ** 2) / 6.0) + 30.0
    shifts = rng.integers(-3, 4, size=(N, 2))
    shifts[0] = 0
    fr = np.stack([np.roll(rng.poisson(base), tuple(s), axis=(0, 1)) for s in shifts]).astype(np.uint16)
    res, G = oracle_mod.iterate_reference(fr, fr[0].astype(np.float32), 1, 1, method="sn", epsilon=eps)
    assert np.array_equal(res.wy, shifts[:, 0]) and np.array_equal(res.wx, shifts[:, 1])
    mean = np.mean([np.roll(f.astype(np.float64), tuple(-s), axis=(0, 1)) for f, s in zip(fr, shifts)], axis=0)
    assert np.max(np.abs(G - np.fft.fft2(mean))) < 1e-9 * np.abs(G[0, 0])
    res2, G2 = oracle_mod.iterate_reference(fr, fr[0].astype(np.float32), 1, 2, method="sn", epsilon=eps)
    for k in range(N):
        S = _sn_direct(fr[k].astype(np.float64), mean, eps)
        assert abs(res2.peak[k] / S.min() - 1) < 1e-11
    assert np.max(np.abs(G2 - G)) < 1e-9 * np.abs(G[0, 0])
