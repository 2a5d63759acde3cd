"""Pins for the oracle's DCT / zigzag / 5-3 DWT. CPU only."""
import itertools

import numpy as np
import pytest
import scipy.fft

import synth


# ---------------------------------------------------------------- zigzag
def test_zigzag_first_six_match_paper(orc, paper_pins):
    want = [tuple(int(t) for t in p.split(",")) for p in paper_pins["zigzag_first6"].split()]
    assert [orc.zigzag(z) for z in range(6)] == want


def test_zigzag_is_a_permutation_and_continues_as_jpeg(orc):
    zz = [orc.zigzag(z) for z in range(64)]
    assert sorted(zz) == sorted(itertools.product(range(8), range(8)))
    assert zz[6:12] == [(0, 3), (1, 2), (2, 1), (3, 0), (4, 0), (3, 1)]
    assert zz[63] == (7, 7) and zz[62] == (7, 6) and zz[61] == (6, 7)
    # neighbours in the scan are neighbours on the grid (a zigzag, not a raster)
    for a, b in zip(zz, zz[1:]):
        assert max(abs(a[0] - b[0]), abs(a[1] - b[1])) == 1


# ---------------------------------------------------------------- DCT 8x8
def test_dct_constant_block_dc_2040(orc, paper_pins):
    X = orc.dct8x8(np.full((8, 8), 255.0))
    assert abs(X[0, 0] - float(paper_pins["dc_bound"])) < 1e-9  # no level shift, orthonormal scaling
    X[0, 0] = 0
    assert np.abs(X).max() < 1e-9
    for cval in [0.0, 1.0, 100.0]:
        assert abs(orc.dct8x8(np.full((8, 8), cval))[0, 0] - 8 * cval) < 1e-9


def test_dct_impulse_closed_form(orc):
    # unit impulse at (i0, j0): X[u][v] = 1/4 C(u)C(v) cos((2 i0+1) u pi/16) cos((2 j0+1) v pi/16)
    for (i0, j0) in [(0, 0), (0, 1), (3, 5), (7, 7), (6, 0)]:
        x = np.zeros((8, 8))
        x[i0, j0] = 1.0
        X = orc.dct8x8(x)
        for u in range(8):
            for v in range(8):
                cu = np.sqrt(0.5) if u == 0 else 1.0
                cv = np.sqrt(0.5) if v == 0 else 1.0
                want = 0.25 * cu * cv * np.cos((2 * i0 + 1) * u * np.pi / 16) * np.cos((2 * j0 + 1) * v * np.pi / 16)
                assert abs(X[u, v] - want) < 1e-12
    x = np.zeros((8, 8)); x[0, 0] = 1.0
    X = orc.dct8x8(x)
    assert abs(X[0, 0] - 0.125) < 1e-12 and abs(X[0, 1] - 0.17337998066526844) < 1e-12


def test_dct_orientation_rows_are_vertical_frequency(orc):
    # an image varying only along x (columns) has energy only in row 0 of X (v = horizontal frequency)
    x = np.tile(np.arange(8, dtype=float)[None, :], (8, 1))
    X = orc.dct8x8(x)
    assert np.abs(X[1:, :]).max() < 1e-9 and abs(X[0, 1]) > 1.0
    # [0,1] (z=1) is the first HORIZONTAL frequency (A3)
    X = orc.dct8x8(x.T)
    assert np.abs(X[:, 1:]).max() < 1e-9 and abs(X[1, 0]) > 1.0


def test_dct_parseval_and_scipy_and_matrix_bruteforce(orc):
    rng = np.random.default_rng(0)
    u = np.arange(8)[:, None]; i = np.arange(8)[None, :]
    Cm = 0.5 * np.cos((2 * i + 1) * u * np.pi / 16)
    Cm[0, :] *= np.sqrt(0.5)
    assert np.allclose(Cm @ Cm.T, np.eye(8), atol=1e-14)  # orthogonality
    for _ in range(50):
        x = rng.integers(0, 256, (8, 8)).astype(float)
        X = orc.dct8x8(x)
        assert abs((x ** 2).sum() - (X ** 2).sum()) < 1e-6 * (x ** 2).sum()          # Parseval
        assert np.abs(X - scipy.fft.dctn(x, norm="ortho")).max() < 1e-9                 # outside library
        assert np.abs(X - Cm @ x @ Cm.T).max() < 1e-9                                   # brute-force matrix product
        assert np.abs(orc.idct8x8(X) - x).max() < 1e-9                                  # inverse
        assert np.abs(orc.idct8x8(X) - scipy.fft.idctn(X, norm="ortho")).max() < 1e-9
    assert np.abs(orc.dct8x8(rng.integers(0, 2, (8, 8)) * 255.0)[0, 1:]).max() <= 1023 + 1e-9  # P:568 AC fits 10 bits


def test_dct_coefficients_layout(orc):
    img = synth.image(24, 16, 3, seed=7)
    coef = orc.dct_coefficients(img)  # [C*nbr*nbc][64] zigzag order
    assert coef.shape == (3 * 2 * 3, 64)
    zz = [orc.zigzag(z) for z in range(64)]
    for c in range(3):
        for br in range(2):
            for bc in range(3):
                X = scipy.fft.dctn(img[8 * br:8 * br + 8, 8 * bc:8 * bc + 8, c].astype(float), norm="ortho")
                b = (c * 2 + br) * 3 + bc
                assert np.abs(coef[b] - np.array([X[r, q] for (r, q) in zz])).max() < 1e-9


def test_energy_compaction_claim(orc):
    # "the DC coefficient ... and another 5 AC coefficients are usually taking over 95% of the energy"
    # statistical sanity on a smooth synthetic image (not a parity pin)
    coef = orc.dct_coefficients(synth.image(64, 64, 1, seed=1, sigma=2.0))
    e = (coef ** 2).sum(axis=0)
    assert e[:6].sum() / e.sum() > 0.95


# ---------------------------------------------------------------- 5/3 lifting DWT
def test_dwt_1d_constant_and_ramp(orc):
    y = orc.dwt53_fwd_1d(np.full(16, 100))
    assert (y[:8] == 100).all() and (y[8:] == 0).all()       # low-pass has DC gain 1 (A12: printed eq. (2) would give 50)
    y = orc.dwt53_fwd_1d(np.arange(0, 32, 2))                # linear ramp -> d = 0 in the interior
    assert (y[8:15] == 0).all()
    assert (y[:7] == np.arange(0, 28, 4)).all()
    # border closed form (A14, x_ext(N) = x(N-2)): d_last = x[N-1] - x[N-2] = 2, s_last = x[N-2] + floor((0 + 2 + 2)/4)
    assert y[15] == 2 and y[7] == 28 + 1


def test_dwt_1d_matches_handwritten_formula(orc):
    # eq. (1) and the A12 reading of eq. (2), retyped with Python's floor division and explicit mirroring
    rng = np.random.default_rng(2)
    for N in [2, 4, 6, 16, 30]:
        x = rng.integers(-128, 128, N)
        xe = lambda i: x[i] if i < N else x[2 * (N - 1) - i]
        d = [xe(2 * n + 1) - (xe(2 * n) + xe(2 * n + 2)) // 2 for n in range(N // 2)]
        de = lambda n: d[n] if n >= 0 else d[-n - 1]   # y_ext(-1) = y(1): d[-1] = d[0]
        s = [x[2 * n] + (de(n - 1) + d[n] + 2) // 4 for n in range(N // 2)]
        y = orc.dwt53_fwd_1d(x)
        assert list(y) == s + d


def test_dwt_1d_equals_53_filter_bank_on_smooth_input(orc):
    # without the floors, lifting equals the Le Gall 5/3 analysis filters: low (-1,2,6,2,-1)/8, high (-1,2,-1)/2
    x = 8 * np.arange(40) ** 2 % 2048  # multiples of 8 keep every floor exact
    x = (x // 8) * 8
    y = orc.dwt53_fwd_1d(x)
    n = np.arange(2, 18)
    hi = x[2 * n + 1] - (x[2 * n] + x[2 * n + 2]) / 2
    lo = (-x[2 * n - 2] + 2 * x[2 * n - 1] + 6 * x[2 * n] + 2 * x[2 * n + 1] - x[2 * n + 2]) / 8
    assert np.abs(y[20 + n] - hi).max() <= 0.5
    assert np.abs(y[n] - lo).max() <= 1.0


def test_dwt_1d_inverse_exact(orc):
    rng = np.random.default_rng(3)
    for N in [2, 4, 8, 64, 250]:
        for _ in range(20):
            x = rng.integers(-128, 128, N)
            assert (orc.dwt53_inv_1d(orc.dwt53_fwd_1d(x)) == x).all()
        for x in [np.full(N, -128), np.full(N, 127), np.where(np.arange(N) % 2, 127, -128)]:
            assert (orc.dwt53_inv_1d(orc.dwt53_fwd_1d(x)) == x).all()


def test_dwt_ranges_match_paper(orc, paper_pins):
    # P:814, input seen as -128..+128: H within +-255.., L within +-192, HH +-511.., LH +-384. Brute force over
    # extreme-valued signals (the extremes of a piecewise-linear map are at the corners of the input cube).
    lo, hi = -128, 128
    maxH = maxL = 0
    for bits in itertools.product([lo, hi], repeat=10):
        y = orc.dwt53_fwd_1d(np.array(bits))
        maxL = max(maxL, np.abs(y[:5]).max()); maxH = max(maxH, np.abs(y[5:]).max())
    assert maxL == int(paper_pins["dwt_range_L"])                       # 192 exactly
    assert int(paper_pins["dwt_range_H"]) <= maxH <= int(paper_pins["dwt_range_H"]) + 1   # 256 for +-128 (paper prints 255)
    # second (vertical) pass on extreme first-pass outputs
    maxHH = maxLH = 0
    for bits in itertools.product([-1, 1], repeat=10):
        b = np.array(bits)
        maxHH = max(maxHH, np.abs(orc.dwt53_fwd_1d(b * maxH)[5:]).max())
        maxLH = max(maxLH, np.abs(orc.dwt53_fwd_1d(b * maxL)[5:]).max())
    assert abs(maxHH - int(paper_pins["dwt_range_HH"])) <= 1 and maxLH == int(paper_pins["dwt_range_LH"])


@pytest.mark.parametrize("L", [1, 2, 3, 4])
def test_dwt_2d_inverse_and_ll_of_constant(orc, L):
    for kind in ["zeros", "ones", "checker", "random", "impulse"]:
        img = synth.special(kind, 48, 32, 1, seed=L)
        planes = orc.dwt_coefficients(img, L)
        rec = orc.dwt_inverse_plane(planes[0], L) + 128
        assert (rec == img[:, :, 0].astype(np.int32)).all()
    planes = orc.dwt_coefficients(np.full((32, 48, 1), 200, dtype=np.uint8), L)
    ll = planes[0, :32 >> L, :48 >> L]
    assert (ll == 200 - 128).all()                     # LL of a constant image = that constant (level-shifted)
    planes[0, :32 >> L, :48 >> L] = 0
    assert (planes == 0).all()


def test_dwt_2d_rows_then_columns(orc):
    # horizontal first, then vertical. Rebuild level 1 from the 1-D routine in that order.
    img = synth.special("random", 16, 8, 1, seed=9)
    x = img[:, :, 0].astype(np.int32) - 128
    rows = np.stack([orc.dwt53_fwd_1d(r) for r in x])
    both = np.stack([orc.dwt53_fwd_1d(c) for c in rows.T]).T
    assert (orc.dwt_coefficients(img, 1)[0] == both).all()
    cols_first = np.stack([orc.dwt53_fwd_1d(c) for c in x.T]).T
    other = np.stack([orc.dwt53_fwd_1d(r) for r in cols_first])
    assert (other != both).any()  # the order matters bit-for-bit (floors), so the test can tell


def test_dwt_ll_fraction(orc, paper_pins):
    assert orc.dwt_private_bytes(64, 64, 1, 2) * int(paper_pins["dwt_ll2_fraction_inv"]) == 64 * 64 * 2  # 1/16
