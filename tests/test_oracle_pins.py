"""Pins for the fp64 oracle (oracle/fdas_oracle.c) against what the paper and the
mathematics fix -- never against the oracle itself or the CUDA path.
Pin numbers P1..P12 follow DESIGN.md / SURVEY.md §8(c)."""
import math

import numpy as np
import pytest
from scipy import special

import oracle
from paper_1511_07343_b200 import synth


# ------------------------------------------------------------------ FFT / spectrum
@pytest.mark.parametrize("n", [1, 2, 8, 64, 1024, 4096])
def test_fft_matches_definition(n):
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    for sign in (-1, +1):
        ref = oracle.dft_direct(x, sign)               # O(n^2) definition, exact phase reduction
        got = oracle.fft(x, sign)
        assert np.max(np.abs(got - ref)) <= 1e-11 * max(1.0, np.max(np.abs(ref)))


def test_dft_direct_is_the_textbook_dft():
    # pin the O(n^2) routine itself: closed forms (delta -> flat, tone -> delta, sign convention)
    n = 16
    d = np.zeros(n, complex); d[3] = 1.0
    k = np.arange(n)
    assert np.allclose(oracle.dft_direct(d, -1), np.exp(-2j * np.pi * 3 * k / n), atol=1e-13)
    tone = np.exp(2j * np.pi * 5 * k / n)
    out = oracle.dft_direct(tone, -1)
    exp = np.zeros(n, complex); exp[5] = n
    assert np.allclose(out, exp, atol=1e-12)


def test_fft_vs_numpy_large():
    rng = np.random.default_rng(7)
    x = rng.standard_normal(1 << 17) + 1j * rng.standard_normal(1 << 17)
    assert np.max(np.abs(oracle.fft(x, -1) - np.fft.fft(x))) < 1e-9
    assert np.max(np.abs(oracle.fft(x, +1) - np.fft.ifft(x) * x.size)) < 1e-9


def test_spectrum_parseval_P8_and_bins():
    N = 1 << 14
    x = synth.make_series(N, 123, [synth.Signal(0.5, 1000.25, 3.0, 0.7)])
    S, mu, raw = oracle.spectrum(x, return_raw=True)
    xd = x.astype(np.float64)
    # P8: |F0|^2 + 2 sum_{1..N/2-1} |Fk|^2 + |F_{N/2}|^2 = N sum x^2
    lhs = abs(raw[0]) ** 2 + 2 * np.sum(np.abs(raw[1:N // 2]) ** 2) + abs(raw[N // 2]) ** 2
    assert lhs == pytest.approx(N * np.sum(xd * xd), rel=1e-12)
    # bins kept are 1..N/2 (G7), DC dropped, Nyquist kept; forward sign e^{-i...} (G6)
    ref = np.fft.rfft(xd)
    assert np.allclose(raw, ref, atol=1e-9)
    assert mu == pytest.approx(np.mean(np.abs(ref[1:]) ** 2), rel=1e-12)
    assert np.allclose(S, ref[1:] / math.sqrt(mu), atol=1e-11)
    assert np.mean(np.abs(S) ** 2) == pytest.approx(1.0, rel=1e-12)
    # real Nyquist bin
    assert abs(S[-1].imag) < 1e-12


def test_spectrum_sign_convention_single_tone():
    # x_n = cos(2 pi k0 n / N): F_k0 = N/2 (real, positive) for the e^{-i} forward transform
    N, k0 = 4096, 37
    n = np.arange(N)
    x = np.cos(2 * np.pi * k0 * n / N + 0.3).astype(np.float32)
    S, mu, raw = oracle.spectrum(x, return_raw=True)
    assert raw[k0] == pytest.approx(N / 2 * np.exp(0.3j), abs=1e-2)   # float32 input rounding


# ------------------------------------------------------------------ response / templates
def fresnel_response(z, d):
    """P2: closed form via Fresnel integrals (scipy convention: fresnel(t) -> (S, C), pi/2 t^2)."""
    if z == 0:
        return np.exp(-1j * np.pi * d) * np.sinc(d)
    if z < 0:                       # P4
        return np.conj(fresnel_response(-z, -d))
    q = -d - z / 2.0
    t0, t1 = q * math.sqrt(2.0 / z), (q + z) * math.sqrt(2.0 / z)
    S1, C1 = special.fresnel(t1)
    S0, C0 = special.fresnel(t0)
    return np.exp(-1j * np.pi * q * q / z) / math.sqrt(2.0 * z) * ((C1 - C0) + 1j * (S1 - S0))


def test_P1_z0_is_sinc_response():
    for d in range(-5, 6):
        r = oracle.response(0.0, d)
        assert abs(r - (1.0 if d == 0 else 0.0)) < 1e-12
    r = oracle.response(0.0, 0.5)
    assert abs(r - (-2j / math.pi)) < 1e-9
    assert abs(r) ** 2 == pytest.approx(0.405284735, abs=1e-8)
    for d in (0.25, -1.5, 2.75):
        assert abs(oracle.response(0.0, d) - np.exp(-1j * np.pi * d) * np.sinc(d)) < 1e-8


def test_P2_fresnel_closed_form():
    worst = 0.0
    for z in (2, 8, 20, 42, 84, 100, -2, -8, -84, 3.7, -55.5):
        for d in (-128, -32, -4, -0.5, 0, 0.5, 1, 5, 31, 42, 127, 127.5, -127.5):
            worst = max(worst, abs(oracle.response(z, d) - fresnel_response(z, d)))
    assert worst < 2e-8


def test_P3_P4_symmetries():
    for z in (2.0, 8.0, 84.0):
        for d in (0, 1, 4, 17):
            a, b = oracle.response(z, d), oracle.response(z, -d)
            assert abs(a - b) < 1e-9                                   # P3: even at integer offsets
            assert abs(oracle.response(-z, d) - np.conj(b)) < 1e-9    # P4
    # P3 general: R_z(d) = e^{-2 pi i d} R_z(-d)
    for d in (0.5, 2.5):
        a, b = oracle.response(8.0, d), oracle.response(8.0, -d)
        assert abs(a - np.exp(-2j * np.pi * d) * b) < 1e-8


def test_P5_worked_values(golden):
    for z, d, re, im in golden("response_values.txt"):
        r = oracle.response(z, d)
        assert abs(r - complex(re, im)) < 2e-8, (z, d, r)


def test_P5_captured_energy_and_layout(golden):
    for m, z, half, energy in golden("captured_energy.txt"):
        m, half = int(m), int(half)
        T = oracle.templates(z, 2.0 * z if z else 1.0, m, interbin=half) if z else oracle.templates(0.0, 1.0, m, interbin=half)
        # z_max = z, dz = 2z -> rows z = -z, +z ; (z = 0: single row)
        nset = 1 + half
        row = T[(T.shape[0] // nset - 1) * nset + half]      # last z row (= +z), requested set
        assert np.sum(np.abs(row) ** 2) == pytest.approx(energy, abs=2e-6)


def test_templates_are_conjugate_responses_with_centred_window():
    m = 64
    T = oracle.templates(20.0, 2.0, m, interbin=1)
    assert T.shape == (42, m)
    # row t = zi*2 + s ; zi = 14 -> z = 8
    for j in (0, 31, 32, 33, 63):
        assert abs(T[14 * 2 + 0, j] - np.conj(fresnel_response(8.0, j - m / 2))) < 2e-8
        assert abs(T[14 * 2 + 1, j] - np.conj(fresnel_response(8.0, j - m / 2 + 0.5))) < 2e-8
    # z = 0 integer template is a delta at tap m/2
    e = np.zeros(m); e[m // 2] = 1.0
    assert np.allclose(T[10 * 2], e, atol=1e-12)


# ------------------------------------------------------------------ correlation
def test_z0_row_is_the_power_spectrum():
    x = synth.make_series(1 << 12, 5)
    S, mu = oracle.spectrum(x)
    T = oracle.templates(4.0, 2.0, 16)
    P = oracle.correlate_direct(S, T)
    assert np.allclose(P[2], np.abs(S) ** 2, rtol=1e-12, atol=1e-14)


def test_direct_sum_against_numpy_convolution():
    # Eq. (1) with arbitrary taps reduces to a library correlation: C[c] = sum_j S[c+j-m/2] T[j]
    rng = np.random.default_rng(3)
    S = rng.standard_normal(300) + 1j * rng.standard_normal(300)
    T = rng.standard_normal((3, 8)) + 1j * rng.standard_normal((3, 8))
    P = oracle.correlate_direct(S, T)
    m = 8
    Sp = np.concatenate([np.zeros(m // 2), S, np.zeros(m)])
    for zi in range(3):
        C = np.array([np.dot(Sp[c:c + m], T[zi]) for c in range(300)])
        assert np.allclose(P[zi], np.abs(C) ** 2, rtol=1e-12)
    # half-bin set reads one bin later (G12)
    T2 = np.repeat(T, 2, axis=0)
    P2 = oracle.correlate_direct(S, T2, interbin=1)
    Sp = np.concatenate([np.zeros(m // 2 - 1), S, np.zeros(m + 1)])
    for zi in range(3):
        C = np.array([np.dot(Sp[c:c + m], T[zi]) for c in range(300)])
        assert np.allclose(P2[zi, 1::2], np.abs(C) ** 2, rtol=1e-12)
        assert np.allclose(P2[zi, 0::2], P[zi], rtol=1e-12)
    # window argument selects columns
    Pw = oracle.correlate_direct(S, T, c0=37, nc=50)
    assert np.array_equal(Pw, P[:, 37:87])


@pytest.mark.parametrize("interbin", [0, 1])
@pytest.mark.parametrize("n,m,L,step", [(1 << 12, 16, 64, None), (1 << 12, 16, 64, 41), (1 << 13, 64, 256, None)])
def test_P9_direct_equals_overlap_save(n, m, L, step, interbin):
    x = synth.make_series(n, 11, [synth.Signal(0.3, n / 8 + 0.37, 5.0, 1.0)])
    S, mu = oracle.spectrum(x)
    T = oracle.templates(8.0, 2.0, m, interbin=interbin)
    Pd = oracle.correlate_direct(S, T, interbin=interbin)
    Pf = oracle.correlate_fft(S, T, L, interbin=interbin, step=step)
    assert Pd.shape == Pf.shape == (9, (n // 2) * (1 + interbin))
    assert np.max(np.abs(Pd - Pf)) <= 1e-10 * np.max(Pd)


def test_P6_P7_config0_noise_free_injection(golden):
    cfg = synth.config(0)
    x = cfg.series(noise=False)
    S, mu = oracle.spectrum(x)
    T = oracle.templates(cfg.z_max, cfg.dz, cfg.width)
    c0, nc = 9999 - 40, 81
    P = oracle.correlate_direct(S, T, c0=c0, nc=nc) * (mu / cfg.n_samples)    # normalise by N instead of mu
    zi, c = np.unravel_index(np.argmax(P), P.shape)
    assert (-20 + 2 * zi, c0 + c + 1) == (8, 10000)                            # z sign (G5), bin<->column (G7)
    rows = {int(z): p for z, b, p in golden("config0_noise_free.txt")}
    for z, p in rows.items():
        assert P[(z + 20) // 2, 9999 - c0] == pytest.approx(p, abs=0.006)
    above = {(int(-20 + 2 * a), int(c0 + b + 1)) for a, b in zip(*np.where(P > 20))}
    assert above == {(z, 10000) for z in rows}
    peak_closed_form = 0.05 ** 2 * cfg.n_samples / 4 * np.sinc(0.3) ** 2
    assert P.max() == pytest.approx(peak_closed_form, rel=2e-4)
    # P6: the plane is the response family |R_{z0-z}(r-r0)|^2 (bow-tie), up to truncation + image leakage
    A2 = (0.05 * cfg.n_samples / 2) ** 2 / cfg.n_samples
    worst = 0.0
    for zi in range(21):
        z = -20 + 2 * zi
        for col in range(9999 - 10, 9999 + 11):
            model = A2 * abs(fresnel_response(8.0 - z, (col + 1) - 10000.3)) ** 2
            worst = max(worst, abs(P[zi, col - c0] - model))
    assert worst < 0.02


def test_P10_noise_statistics():
    x = synth.make_series(1 << 16, 99)
    S, mu = oracle.spectrum(x)
    assert mu == pytest.approx(1 << 16, rel=0.02)                # unit-variance noise: mu ~ N
    T = oracle.templates(20.0, 2.0, 64)
    P = oracle.correlate_fft(S, T, 1024)
    energy = np.sum(np.abs(T) ** 2, axis=1)
    assert np.allclose(P.mean(axis=1), energy, rtol=0.03)        # each row has mean sum|T|^2 (~1)
    frac = np.mean(P[10] > 3.0)                                   # z=0 row: P ~ Exp(1)
    assert frac == pytest.approx(math.exp(-3.0), rel=0.1)


def test_P11_interbin_tone():
    N, k0 = 1 << 12, 700
    n = np.arange(N)
    x = np.cos(2 * np.pi * (k0 + 0.5) * n / N)
    F = np.fft.rfft(x)[1:] / (N / 2)            # unit tone amplitude, bins 1..N/2 (no mean-power normalisation here)
    T = oracle.templates(0.0, 1.0, 256, interbin=1)
    P = oracle.correlate_direct(F, T, interbin=1, c0=k0 - 3, nc=6)
    col_k0 = (k0 - 1) - (k0 - 3)
    assert P[0, 2 * col_k0] == pytest.approx(0.405285, abs=2e-4)          # integer column at bin k0
    assert P[0, 2 * (col_k0 + 1)] == pytest.approx(0.405285, abs=2e-4)    # integer column at bin k0+1
    assert P[0, 2 * col_k0 + 1] == pytest.approx(0.996836, abs=3e-4)      # half column r = k0 + 1/2


# ------------------------------------------------------------------ candidates / harmonic sum
def test_candidates_strict_threshold():
    P = np.array([[1.0, 20.0, 20.0000001], [25.0, 3.0, 19.9]])
    c = oracle.candidates(P, 20.0)
    assert [(int(r["col"]), int(r["zi"]), int(r["nharm"])) for r in c] == [(2, 0, 1), (0, 1, 1)]
    assert c["power"][1] == 25.0


def test_thresholds_P12(golden):
    assert oracle.threshold(1) == pytest.approx(-math.log(1e-6), abs=1e-10)
    for H, T in golden("thresholds.txt"):
        got = oracle.threshold(int(H))
        assert got == pytest.approx(T, abs=2e-9)
        assert special.gammaincc(int(H), got) == pytest.approx(1e-6, rel=1e-9)   # library survival function


def py_round_half_up(a, h, H):
    return (a * h + H // 2) // H


def brute_harmsum(P, bin0, max_harm):
    """Pure-python restatement of the O6 definition (tiny planes only)."""
    n_z, n_cols = P.shape
    zc = (n_z - 1) // 2
    out = {}
    H = 1
    while H <= max_harm:
        S = np.zeros_like(P)
        for zi in range(n_z):
            zeta = zi - zc
            for c in range(n_cols):
                k = bin0 + c
                acc = 0.0
                for h in range(1, H + 1):
                    kh = py_round_half_up(k, h, H)
                    zh = int(math.copysign(py_round_half_up(abs(zeta), h, H), zeta)) if zeta else 0
                    if kh >= bin0:
                        acc += P[zc + zh, kh - bin0]
                S[zi, c] = acc
        out[H] = S
        H *= 2
    return out


def test_harmsum_brute_force_toy_plane_P12():
    rng = np.random.default_rng(12)
    P = rng.exponential(1.0, size=(9, 256))
    thr = oracle.thresholds(16, 1e-2)
    cands, S = oracle.harmsum(P, 16, thr, bin0=1, return_sums=True)
    ref = brute_harmsum(P, 1, 16)
    for s, H in enumerate((1, 2, 4, 8, 16)):
        assert np.allclose(S[s], ref[H], rtol=1e-13)
    want = {(H, zi, c) for s, H in enumerate((1, 2, 4, 8, 16)) for zi, c in zip(*np.where(ref[H] > thr[s]))}
    got = {(int(r["nharm"]), int(r["zi"]), int(r["col"])) for r in cands}
    assert got == want and len(cands) == len(want)


def test_harmsum_constant_plane_and_rounding_P12():
    P = np.ones((11, 400))
    _, S = oracle.harmsum(P, 16, np.full(5, 1e9), bin0=1, return_sums=True)
    for s, H in enumerate((1, 2, 4, 8, 16)):
        # all k_h >= bin0  <=>  round(k/H) >= 1  <=>  k >= H/2 (round half up)
        k = 1 + np.arange(400)
        full = k >= max(1, H // 2)
        assert np.all(S[s][:, full] == H)
    # exact ties: odd k with h/H = 1/2 rounds UP (k=5 -> 3), zeta ties away from zero (+-3 -> +-2)
    P = np.zeros((11, 64)); P[5 + 2, 3 - 1] = 7.0; P[5 - 2, 3 - 1] = 9.0
    _, S = oracle.harmsum(P, 2, np.full(2, 1e9), bin0=1, return_sums=True)
    assert S[1][5 + 3, 5 - 1] == 7.0 and S[1][5 - 3, 5 - 1] == 9.0
    assert S[1][5 + 4, 5 - 1] == 7.0 and S[1][5 + 4, 6 - 1] == 7.0     # zeta 4 -> 2 ; k 6 -> 3
    assert S[1][5 + 5, 5 - 1] == 0.0                                     # zeta 5 -> 3 (away from zero)


def test_harmsum_single_bright_cell_preimages_P12():
    n_z, n_cols, bin0 = 21, 512, 1
    zc = 10
    kstar, zstar = 97, 3
    P = np.zeros((n_z, n_cols)); P[zc + zstar, kstar - bin0] = 100.0
    cands = oracle.harmsum(P, 16, np.full(5, 50.0), bin0=bin0)
    got = {(int(r["nharm"]), int(r["zi"]) - zc, int(r["col"]) + bin0) for r in cands}
    want = set()
    for H in (1, 2, 4, 8, 16):
        for zeta in range(-zc, zc + 1):
            for k in range(bin0, bin0 + n_cols):
                hit = 0
                for h in range(1, H + 1):
                    kh = (k * h + H // 2) // H
                    zh = (abs(zeta) * h + H // 2) // H * (1 if zeta >= 0 else -1)
                    hit += (kh == kstar and zh == zstar)
                if hit:
                    want.add((H, zeta, k))
    assert got == want


def test_harmsum_stage_nesting_identity():
    # S_2H = S_H + odd-h terms of stage 2H (the rounding rule is invariant under (h,H)->(2h,2H))
    rng = np.random.default_rng(5)
    P = rng.exponential(1.0, size=(7, 300))
    _, S = oracle.harmsum(P, 8, np.full(4, 1e9), return_sums=True)
    assert np.all(S[1] >= S[0]) and np.all(S[2] >= S[1]) and np.all(S[3] >= S[2])
    assert np.allclose(S[0], P)


def test_P13_harmsum_of_a_noise_free_pulse_train():
    """End-to-end pin of the harmonic-sum reading G16: (k, zeta) label the TOP
    harmonic, and both the bin and the z index are stretched by h/H.  A noise-free train with harmonics
    h = 1..4 of a fundamental at bin r0 = 300 drifting z0 = 2 bins puts its h-th harmonic at (h r0, h z0)
    ("pulse harmonics", z scales with the frequency).  By P6 the plane peaks there
    at (A_h N/2)^2 / mu, so the closed form is
        S_H(H r0, H z0) = sum_{h<=H} (A_h N/2)^2 / mu,
    it is the global maximum of stage H, and the fundamental-labelled reading (sums placed at (r0, z0))
    finds only the h = 1 peak."""
    N, r0, z0 = 1 << 14, 300, 2
    amps = [1.0, 0.8, 0.6, 0.5]
    sig = [synth.Signal(a, r0 * (h + 1), z0 * (h + 1), 0.3 * h) for h, a in enumerate(amps)]
    x = synth.make_series(N, 1, sig, noise=False)
    S, mu = oracle.spectrum(x)
    T = oracle.templates(8.0, 2.0, 64)
    P = oracle.correlate_fft(S, T, 1024)
    peak = [(a * N / 2) ** 2 / mu for a in amps]
    zi = lambda z: int((z + 8) // 2)
    for h in range(4):                                           # P6 at each harmonic: the plane itself
        assert P[zi(z0 * (h + 1)), r0 * (h + 1) - 1] == pytest.approx(peak[h], rel=2e-3)
    thr = np.array([1e30, 1e30, 1e30])
    _, sums = oracle.harmsum(P, 4, thr, bin0=1, return_sums=True)
    for st, H in enumerate((1, 2, 4)):
        want = sum(peak[:H])
        got = sums[st][zi(z0 * H), r0 * H - 1]
        assert got == pytest.approx(want, rel=2e-3), (H, got, want)
        if H > 1:
            assert np.unravel_index(np.argmax(sums[st]), sums[st].shape) == (zi(z0 * H), r0 * H - 1)
    # fundamental labelling would look at (r0, z0) and see one harmonic only
    assert sums[2][zi(z0), r0 - 1] < 1.05 * peak[0]


def test_all_zero_series_gives_zero_spectrum_G22():
    """Degenerate input (reading G22): mu = 0 -> S := 0, not 0/0."""
    S, mu = oracle.spectrum(np.zeros(1 << 10, np.float32))
    assert mu == 0.0 and not np.any(S)


# ------------------------------------------------------------------ time-domain resampling (G23)
def test_resample_identity_and_nearest_sample_property():
    N = 1 << 12
    x = np.arange(N, dtype=np.float32)                  # y then holds the chosen source index itself
    assert np.array_equal(oracle.resample(x, 0.0), x)
    for beta in (0.3, -0.2, 1e-4):
        n = oracle.resample(x, beta).astype(np.int64)
        assert np.all(np.diff(n) >= 0) and n[0] == 0    # monotone map that starts at the first sample
        # the chosen sample is the nearest to the exact solution of u + beta (u^2 - u) = m/N (evaluated in
        # extended precision from the defining equation, not from the oracle's root formula)
        m = np.arange(N, dtype=np.longdouble)
        g = lambda nn: (nn / N + np.longdouble(beta) * ((nn / N) ** 2 - nn / N)) * N      # forward map, in samples
        d0 = np.abs(g(n.astype(np.longdouble)) - m)
        ok = n < N - 1                                   # the last sample is a clamp, not a nearest sample
        assert np.all(d0[ok] <= np.abs(g(n + 1.0) - m)[ok] + 1e-9)
        assert np.all(d0[n > 0] <= np.abs(g(n - 1.0) - m)[n > 0] + 1e-9)
    with pytest.raises(ValueError):
        oracle.resample(x, 0.5)


def test_resample_turns_an_accelerated_sinusoid_into_a_tone():
    """PAPER.md:17 in one number: a noise-free sinusoid of mean frequency r0 = 3000 drifting z = 24 bins,
    resampled at beta = z/(2 r0), is a pure tone at bin r0: all of A^2 N/4 (here normalised by mu) comes back in
    one bin, as for an unaccelerated tone, while the raw series leaves a few per cent there.  The FDAS plane
    of the RAW series has the same power at (r0, z) -- the two searches cross-check each other."""
    N, r0, z, A = 1 << 16, 3000, 24, 1.0
    x = synth.make_series(N, 1, [synth.Signal(A, r0, z, 0.7)], noise=False)
    S_raw, mu_raw = oracle.spectrum(x)
    y = oracle.resample(x, z / (2.0 * r0))
    S_y, mu_y = oracle.spectrum(y)
    full = (A * N / 2) ** 2                              # |F_r0|^2 of a pure tone
    p_y = abs(S_y[r0 - 1]) ** 2 * mu_y
    assert p_y == pytest.approx(full, rel=0.02) and int(np.argmax(np.abs(S_y))) == r0 - 1
    assert abs(S_raw[r0 - 1]) ** 2 * mu_raw < 0.2 * full
    T = oracle.templates(24.0, 2.0, 64)
    P = oracle.correlate_direct(S_raw, T, c0=r0 - 33, nc=64)
    zi, c = np.unravel_index(np.argmax(P), P.shape)
    assert (zi, c + r0 - 33) == (24, r0 - 1)             # row of z = +24, the column of bin r0
    assert P[zi, c] * mu_raw == pytest.approx(full, rel=0.02)
