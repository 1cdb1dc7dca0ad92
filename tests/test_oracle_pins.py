"""Pins for the CPU oracle (oracle/), CPU only.

Each test checks the oracle against something other than itself: hand-worked values
(tests/golden/handworked.txt), closed forms, an independent numpy full-matrix brute force, structural
invariants and O(N*T) integer identities ("What pins each part").
"""
from pathlib import Path

import numpy as np
import pytest

import oracle
import workloads as wl

GOLDEN = Path(__file__).parent / "golden" / "handworked.txt"


def _tri(n):
    return n * (n + 1) // 2


def _both(frame):
    """naive and planar must agree bit for bit; return the common value."""
    a = oracle.naive(frame)
    b = oracle.planar(frame)
    assert a.dtype == np.int32 and b.dtype == np.int32
    np.testing.assert_array_equal(a, b)
    return a


# ---------------------------------------------------------------- hand-worked golden values
def _golden_cases():
    cases = []
    for ln in GOLDEN.read_text().splitlines():
        ln = ln.strip()
        if not ln or ln.startswith("#"):
            continue
        head, data, exp = [s.strip() for s in ln.split("|")]
        t, n = map(int, head.split())
        b = np.array([int(x, 16) for x in data.split()], dtype=np.uint8).reshape(t, 1, n)
        e = np.array([[int(v) for v in p.split(",")] for p in exp.split()], dtype=np.int64)
        cases.append((ln, b, e))
    return cases


@pytest.mark.parametrize("line,frame,expected", _golden_cases(), ids=lambda v: v if isinstance(v, str) else None)
def test_handworked(line, frame, expected):
    got = _both(frame)
    assert got.shape == (1, _tri(frame.shape[2]), 2)
    np.testing.assert_array_equal(got[0], expected)
    # the same pencil values through the numpy statement and the sampled-pairs entry point
    vre, vim = oracle.brute_full(frame)
    np.testing.assert_array_equal(oracle.triangle_from_full(vre, vim)[0], expected)


def test_golden_file_has_cases():
    assert len(_golden_cases()) >= 8


# ---------------------------------------------------------------- output size / pair indexing
def test_table1_output_size():
    # PAPER.md:142 Table I "Output Data (10s Cadence) 16.8": 64 ch x 32896 pairs x 8 B = 16,842,752 B,
    # x16 servers = 269.5 MB -> upper triangle INCLUDING autos, 2 x 32-bit per pair.
    assert oracle.n_pairs(256) == 32896
    assert 64 * oracle.n_pairs(256) * 8 == 16_842_752
    assert round(16 * 16_842_752 / 1e6, 1) == 269.5
    assert wl.CONFIGS["C2"].output_bytes == 16_842_752
    assert oracle.n_pairs(16) == 136  # BASELINE.json:configs[0]


def test_pair_index_corners_and_bijection():
    n = 16
    assert oracle.pair_index(n, 0, 0) == 0
    assert oracle.pair_index(n, 0, n - 1) == 15
    assert oracle.pair_index(n, 1, 1) == 16
    assert oracle.pair_index(n, n - 1, n - 1) == 135
    for n in (1, 2, 3, 16, 37):
        seen = [oracle.pair_index(n, i, j) for i in range(n) for j in range(i, n)]
        assert seen == list(range(_tri(n)))  # row-major order, no gaps


@pytest.mark.parametrize("n", [5, 16])
def test_one_hot_and_two_hot(n):
    t, f = 7, 2
    for k in (0, n // 2, n - 1):
        fr = np.zeros((t, f, n), np.uint8)
        fr[:, 1, k] = wl.pack(3, -2)
        v = _both(fr)
        assert np.count_nonzero(v[0]) == 0  # channel 0 silent
        nz = np.argwhere(v[1] != 0)
        assert nz.tolist() == [[oracle.pair_index(n, k, k), 0]]
        assert v[1, oracle.pair_index(n, k, k), 0] == t * 13
    a, b = 1, n - 2
    fr = np.zeros((t, f, n), np.uint8)
    fr[:, 0, a] = wl.pack(1, 2)    # 1+2i
    fr[:, 0, b] = wl.pack(-3, 1)   # -3+i ; (1+2i)*conj(-3+i) = (1+2i)(-3-i) = -3 -i -6i +2 = -1-7i
    v = _both(fr)
    rows = sorted(set(np.argwhere(v[0] != 0)[:, 0].tolist()))
    assert rows == sorted([oracle.pair_index(n, a, a), oracle.pair_index(n, a, b), oracle.pair_index(n, b, b)])
    np.testing.assert_array_equal(v[0, oracle.pair_index(n, a, b)], [-1 * t, -7 * t])
    np.testing.assert_array_equal(v[0, oracle.pair_index(n, a, a)], [5 * t, 0])
    np.testing.assert_array_equal(v[0, oracle.pair_index(n, b, b)], [10 * t, 0])


# ---------------------------------------------------------------- closed forms
@pytest.mark.parametrize("byte", [0x00, 0x88, 0x7F, 0x8F, 0x31, 0xF8])
def test_constant_input_closed_form(byte):
    n, f, t = 6, 3, 50
    re, im = oracle.unpack(np.array([byte], np.uint8))
    mag2 = int(re[0] ** 2 + im[0] ** 2)
    v = _both(wl.constant_frame(n, f, t, byte))
    assert (v[:, :, 0] == t * mag2).all() and (v[:, :, 1] == 0).all()


def test_unpack_table_all_256_bytes():
    # R2/R3 written out independently: nibble value v -> v if v < 8 else v - 16
    b = np.arange(256, dtype=np.uint8)
    re, im = oracle.unpack(b)
    for x in range(256):
        hi, lo = x >> 4, x & 15
        assert re[x] == (hi if hi < 8 else hi - 16)
        assert im[x] == (lo if lo < 8 else lo - 16)
    assert re.min() == -8 and re.max() == 7 and im.min() == -8 and im.max() == 7
    # and the C decode agrees on every byte: auto of a single sample = re^2 + im^2
    v = oracle.naive(b.reshape(1, 256, 1))
    np.testing.assert_array_equal(v[:, 0, 0], re ** 2 + im ** 2)
    # pack is the inverse of the decode
    np.testing.assert_array_equal(wl.pack(re, im), b)


def test_int32_stress_bound_exact():
    # max |sum| = 128*T (BASELINE.json:configs[4]); T = 2^20 -> 2^27 exactly, well inside int32
    t = 1 << 20
    v = oracle.planar(wl.constant_frame(2, 1, t, 0x88))
    assert (v[0, :, 0] == 128 * t).all() and (v[0, :, 1] == 0).all()


def test_int32_overflow_is_reported_not_wrapped():
    t = (1 << 24)  # 128 * 2^24 = 2^31 > INT32_MAX
    fr = wl.constant_frame(1, 1, t, 0x88)
    with pytest.raises(OverflowError):
        oracle.naive(fr)
    with pytest.raises(OverflowError):
        oracle.planar(fr)
    v = oracle.planar(fr[: t - 1])
    assert v[0, 0, 0] == 128 * (t - 1)


# ---------------------------------------------------------------- brute force full N x N
@pytest.mark.parametrize("n,f,t,seed", [(16, 4, 256, 0), (3, 1, 1, 1), (7, 2, 33, 2), (32, 3, 65, 3), (1, 1, 5, 4)])
def test_against_numpy_full_matrix(n, f, t, seed):
    fr = wl.uniform_frame(n, f, t, seed)
    v = _both(fr)
    vre, vim = oracle.brute_full(fr)
    np.testing.assert_array_equal(v, oracle.triangle_from_full(vre, vim))
    # Hermitian structure of the brute-force matrix: V[j,i] = conj(V[i,j]); autos real and >= 0
    np.testing.assert_array_equal(vre, vre.transpose(0, 2, 1))
    np.testing.assert_array_equal(vim, -vim.transpose(0, 2, 1))
    d = np.arange(n)
    assert (vim[:, d, d] == 0).all() and (vre[:, d, d] >= 0).all()
    # third, fully independent statement: complex128 arithmetic is exact at these magnitudes
    re, im = oracle.unpack(fr)
    x = re + 1j * im
    vc = np.einsum("tfi,tfj->fij", x, x.conj())
    np.testing.assert_array_equal(vre, np.rint(vc.real).astype(np.int64))
    np.testing.assert_array_equal(vim, np.rint(vc.imag).astype(np.int64))


def test_c1_config_shape_and_autos():
    c = wl.CONFIGS["C1"]
    fr = c.frame()
    assert fr.shape == (256, 4, 16) and fr.nbytes == 16384
    v = _both(fr)
    assert v.shape == (4, 136, 2)
    re, im = oracle.unpack(fr)
    for i in range(16):
        np.testing.assert_array_equal(v[:, oracle.pair_index(16, i, i), 0], (re[:, :, i] ** 2 + im[:, :, i] ** 2).sum(0))


# ---------------------------------------------------------------- layout / strides / channels
def test_channel_independence_and_permutation():
    n, f, t = 8, 5, 40
    fr = wl.uniform_frame(n, f, t, 11)
    v = _both(fr)
    perm = np.array([3, 0, 4, 1, 2])
    np.testing.assert_array_equal(_both(np.ascontiguousarray(fr[:, perm, :])), v[perm])
    only = np.zeros_like(fr)
    only[:, 2, :] = fr[:, 2, :]
    vo = _both(only)
    np.testing.assert_array_equal(vo[2], v[2])
    assert np.count_nonzero(vo[[0, 1, 3, 4]]) == 0


def test_stride_pattern_frame():
    # byte depends on (t, f, n) through distinct moduli: any stride mix-up changes the answer
    n, f, t = 6, 4, 30
    tt, ff, nn = np.meshgrid(np.arange(t), np.arange(f), np.arange(n), indexing="ij")
    fr = wl.pack((tt * 3 + ff * 5 + nn * 7) % 16 - 8, (tt + ff * 2 + nn * 11) % 16 - 8)
    v = _both(fr)
    vre, vim = oracle.brute_full(fr)
    np.testing.assert_array_equal(v, oracle.triangle_from_full(vre, vim))
    assert fr.tobytes() != np.ascontiguousarray(fr.transpose(0, 2, 1)).tobytes()


def test_input_permutation_equivariance():
    n, f, t = 9, 2, 25
    fr = wl.uniform_frame(n, f, t, 5)
    vre, vim = oracle.brute_full(fr)
    perm = np.random.default_rng(6).permutation(n)
    v2 = _both(np.ascontiguousarray(fr[:, :, perm]))
    for ch in range(f):
        for i in range(n):
            for j in range(i, n):
                p = oracle.pair_index(n, i, j)
                a, b = perm[i], perm[j]
                assert v2[ch, p, 0] == vre[ch, a, b]
                assert v2[ch, p, 1] == vim[ch, a, b]  # full matrix already holds the conjugate when a > b


# ---------------------------------------------------------------- time axis: linearity, order, padding
def test_linearity_over_split_frames_and_time_permutation():
    n, f, t = 10, 3, 64
    fr = wl.uniform_frame(n, f, t, 21)
    v = _both(fr).astype(np.int64)
    a, b = fr[:17], fr[17:]
    np.testing.assert_array_equal(_both(np.ascontiguousarray(a)).astype(np.int64) + _both(np.ascontiguousarray(b)), v)
    perm = np.random.default_rng(3).permutation(t)
    np.testing.assert_array_equal(_both(np.ascontiguousarray(fr[perm])), v)


def test_zero_padding_is_exact():
    # lost packets are zero-filled: such points just hold fewer samples
    n, f, t = 6, 2, 20
    fr = wl.uniform_frame(n, f, t, 8)
    v = _both(fr)
    more_t = np.concatenate([fr, np.zeros((13, f, n), np.uint8)], axis=0)
    np.testing.assert_array_equal(_both(more_t), v)
    more_n = np.concatenate([fr, np.zeros((t, f, 4), np.uint8)], axis=2)
    v2 = _both(np.ascontiguousarray(more_n))
    for i in range(n):
        for j in range(i, n):
            np.testing.assert_array_equal(v2[:, oracle.pair_index(n + 4, i, j)], v[:, oracle.pair_index(n, i, j)])
    for i in range(n + 4):
        for j in range(max(i, n), n + 4):
            assert not v2[:, oracle.pair_index(n + 4, i, j)].any()


def test_empty_time_axis():
    v = _both(np.zeros((0, 2, 4), np.uint8))
    assert v.shape == (2, 10, 2) and not v.any()


# ---------------------------------------------------------------- global symmetries
def test_symmetries_negate_rotate_conjugate():
    n, f, t = 8, 2, 50
    rng = np.random.default_rng(9)
    re = rng.integers(-7, 8, size=(t, f, n))  # avoid -8 so that -x and i*x stay representable
    im = rng.integers(-7, 8, size=(t, f, n))
    v = _both(wl.pack(re, im))
    np.testing.assert_array_equal(_both(wl.pack(-re, -im)), v)        # x -> -x
    np.testing.assert_array_equal(_both(wl.pack(-im, re)), v)         # x -> i*x
    vc = _both(wl.pack(re, -im))                                      # x -> conj(x)
    np.testing.assert_array_equal(vc[:, :, 0], v[:, :, 0])
    np.testing.assert_array_equal(vc[:, :, 1], -v[:, :, 1])
    # swapping nibbles == conjugating V (SURVEY.md 8(c) point 2)
    vs = _both(wl.pack(im, re))
    np.testing.assert_array_equal(vs[:, :, 0], v[:, :, 0])
    np.testing.assert_array_equal(vs[:, :, 1], -v[:, :, 1])


# ---------------------------------------------------------------- O(N*T) identities (used at full size on the GPU side)
def test_total_power_and_freivalds_identities():
    n, f, t = 24, 3, 100
    fr = wl.gaussian_frame(n, f, t, 31)
    v = _both(fr)
    np.testing.assert_array_equal(oracle.lhs_total_power(v, n), oracle.identity_total_power(fr))
    rng = np.random.default_rng(1)
    for ch in range(f):
        for _ in range(3):
            u = rng.integers(-3, 4, size=n)
            w = rng.integers(-3, 4, size=n)
            assert oracle.freivalds_lhs(v[ch], n, u, w) == oracle.freivalds_rhs(fr[:, ch, :], u, w)
    # the identities do catch a single wrong entry
    bad = v.copy()
    bad[1, oracle.pair_index(n, 3, 17), 1] += 1
    u = np.zeros(n, np.int64); u[3] = 1
    w = np.zeros(n, np.int64); w[17] = 1
    assert oracle.freivalds_lhs(bad[1], n, u, w) != oracle.freivalds_rhs(fr[:, 1, :], u, w)
    bad = v.copy()
    bad[2, oracle.pair_index(n, 0, 5), 0] -= 1
    assert (oracle.lhs_total_power(bad, n) != oracle.identity_total_power(fr)).any()


def test_pairs_entry_point_matches_full():
    n, f, t = 12, 4, 77
    fr = wl.uniform_frame(n, f, t, 13)
    v = _both(fr)
    idx = np.array([[ch, i, j] for ch in range(f) for i in range(n) for j in range(i, n)], np.int32)
    got = oracle.pairs(fr, idx)
    np.testing.assert_array_equal(got.reshape(f, -1, 2), v)
    with pytest.raises(ValueError):
        oracle.pairs(fr, np.array([[0, 5, 2]], np.int32))  # i > j is not a stored pair


def test_planar_channel_range():
    fr = wl.uniform_frame(8, 5, 30, 2)
    v = _both(fr)
    part = oracle.planar(fr, 1, 3)
    np.testing.assert_array_equal(part[1:3], v[1:3])
    assert not part[[0, 3, 4]].any()


# ---------------------------------------------------------------- generators (statistical)
def test_gaussian_generator_statistics():
    from math import erf, sqrt
    fr = wl.gaussian_frame(64, 8, 2048, 2)
    re, im = oracle.unpack(fr)
    x = np.concatenate([re.ravel(), im.ravel()])
    phi = lambda z: 0.5 * (1 + erf(z / sqrt(2)))
    pmf = {k: phi((k + 0.5) / 2.5) - phi((k - 0.5) / 2.5) for k in range(-7, 7)}
    pmf[-8] = phi(-7.5 / 2.5)
    pmf[7] = 1 - phi(6.5 / 2.5)
    assert abs(sum(pmf.values()) - 1) < 1e-12
    n = x.size
    for k, p in pmf.items():
        assert abs((x == k).mean() - p) < 6 * sqrt(p * (1 - p) / n) + 1e-6
    ex2 = sum(k * k * p for k, p in pmf.items())
    assert abs(ex2 - 6.298) < 0.01          # SURVEY.md 8(c) "Generators"
    assert abs((x.astype(np.float64) ** 2).mean() - ex2) < 0.02
    # autos ~ 2*E[x^2]*T
    v = oracle.planar(fr[:, :1, :8].copy())
    autos = np.array([v[0, oracle.pair_index(8, i, i), 0] for i in range(8)])
    assert np.all(np.abs(autos / 2048 - 2 * ex2) < 0.6)


def test_sky_generator_has_positive_offdiagonal_mean():
    fr = wl.gaussian_frame(16, 2, 4096, 4, sigma_sky=1.0)
    v = oracle.planar(fr)
    off = np.array([v[0, oracle.pair_index(16, i, j), 0] for i in range(16) for j in range(i + 1, 16)])
    assert 1.5 < off.mean() / 4096 < 2.5     # ~ 2*sigma_sky^2 per sample


def test_stress_generator_layout():
    fr = wl.stress_frame(8, 2, 64, 5)
    assert (fr[:, :, :4] == 0x88).all()
    assert len(np.unique(fr[:, :, 4:])) > 50
    v = oracle.planar(fr)
    for i in range(4):
        for j in range(i, 4):
            np.testing.assert_array_equal(v[:, oracle.pair_index(8, i, j)], [[128 * 64, 0]] * 2)
    # const-random pairs: V[i,j] = c * conj(sum_t x_j), c = -8-8i
    re, im = oracle.unpack(fr)
    for j in range(4, 8):
        sr, si = re[:, 0, j].sum(), im[:, 0, j].sum()
        # (-8-8i)(sr - i si) = -8 sr - 8 si + i(8 si - 8 sr)
        np.testing.assert_array_equal(v[0, oracle.pair_index(8, 0, j)], [-8 * sr - 8 * si, 8 * si - 8 * sr])


def test_generators_are_seeded():
    for kind in ("uniform", "gaussian", "gaussian_sky", "stress"):
        a = wl.make_frame(kind, 16, 2, 40, 7)
        b = wl.make_frame(kind, 16, 2, 40, 7)
        c = wl.make_frame(kind, 16, 2, 40, 8)
        assert a.tobytes() == b.tobytes() and a.tobytes() != c.tobytes()
