"""Reading A20: the large-V tensor-core products take their operands as FP16 hi/lo pairs with
power-of-two scales instead of TF32 pairs.  These checks are plain numpy (no GPU, no library code): they pin
the arithmetic claims the reading rests on -- the same 11-bit significand, the scale rule, no overflow, and
the size of what a three-product split drops."""
import numpy as np


def split16(v):
    hi = v.astype(np.float16)
    lo = (v - hi.astype(np.float64)).astype(np.float16)
    return hi.astype(np.float64), lo.astype(np.float64)


def tf32_rna(v):
    """round-to-nearest-away to 10 explicit mantissa bits, as cvt.rna.tf32.f32 does on an FP32 value"""
    u = v.astype(np.float32).view(np.uint32).astype(np.uint64)
    u = (u + 0x1000) & 0xFFFFE000
    return u.astype(np.uint32).view(np.float32).astype(np.float64)


def scale_of(maxabs, top):
    return 2.0 ** (top - int(np.floor(np.log2(maxabs))))


def test_fp16_and_tf32_significands_are_the_same_width():
    rng = np.random.default_rng(1)
    v = rng.uniform(1.0, 2.0, 100000)
    e16 = np.abs(v - v.astype(np.float16).astype(np.float64)) / v
    e32 = np.abs(v - tf32_rna(v)) / v
    assert e16.max() <= 2.0 ** -11 and e32.max() <= 2.0 ** -11
    assert e16.max() > 2.0 ** -12.1 and e32.max() > 2.0 ** -12.1       # both really are 11 bits


def test_scaled_split_of_the_factor():
    """s Lc entries over ten orders of magnitude: hi + lo reproduces c v to 2^-22 |v| where lo is a normal
    number, and to 2^-37 of the largest entry below that; nothing overflows."""
    rng = np.random.default_rng(2)
    for maxabs in (3e-5, 0.037, 1.0, 812.0):
        v = maxabs * np.concatenate([[1.0, -1.0], rng.uniform(-1, 1, 20000) * 10.0 ** rng.uniform(-10, 0, 20000)])
        c = scale_of(maxabs, 12)
        assert 2.0 ** 12 <= c * maxabs < 2.0 ** 13
        hi, lo = split16(c * v)
        assert np.all(np.isfinite(hi)) and np.abs(hi).max() < 65504
        err = np.abs(c * v - hi - lo) / c
        big = np.abs(c * v) >= 2.0 ** -14 * 2.0 ** 11                  # lo is a normal FP16 number
        assert np.all(err[big] <= 2.0 ** -22 * np.abs(v[big]))
        assert np.all(err <= np.maximum(2.0 ** -22 * np.abs(v), 2.0 ** -37 * maxabs))


def test_scaled_split_of_the_normals():
    rng = np.random.default_rng(3)
    z = np.concatenate([rng.standard_normal(200000), [6.66, -6.66, 1e-4, 0.0]])
    hi, lo = split16(8.0 * z)
    assert np.abs(hi).max() < 65504
    err = np.abs(8.0 * z - hi - lo) / 8.0
    assert np.all(err <= np.maximum(2.0 ** -22 * np.abs(z), 2.0 ** -28))   # 2^-25 scaled, / 8


def test_three_product_split_drops_only_lo_lo():
    """d = sum_y L_xy z_y from hi*hi + hi*lo + lo*hi in exact arithmetic: the error is the lo*lo term plus the
    representation error of the pairs, ~2^-21 of sum |L||z| -- the same bound as 3xTF32."""
    rng = np.random.default_rng(4)
    V = 512
    Lc = np.tril(rng.standard_normal((V, V)) * 0.037 * np.exp(-np.abs(np.subtract.outer(np.arange(V), np.arange(V))) / 20.0))
    z = rng.standard_normal(V)
    c = scale_of(np.abs(Lc).max(), 12)
    Lh, Ll = split16(c * Lc)
    zh, zl = split16(8.0 * z)
    d = (Lh @ zh + Lh @ zl + Ll @ zh) / (8.0 * c)
    ref = Lc @ z
    bound = 2.0 ** -20 * (np.abs(Lc) @ np.abs(z))
    assert np.all(np.abs(d - ref) <= bound)
    Th, Tl = tf32_rna(Lc), tf32_rna(Lc - tf32_rna(Lc))
    yh = tf32_rna(z)
    yl = z - yh
    d32 = Th @ yh + Th @ yl + Tl @ yh
    assert np.all(np.abs(d32 - ref) <= bound)


def test_covariance_operand_scale_from_the_per_site_bound():
    """amax_x = max_i |phi_xi| + |mu_x| bounds |phi_xi - mu_x|; c = 2^(11 - e) keeps c (phi - mu) below 2^12."""
    rng = np.random.default_rng(5)
    phi = rng.standard_normal((64, 4096)) * rng.uniform(0.1, 30.0, (64, 1)) + rng.uniform(-50, 50, (64, 1))
    mu = phi.mean(axis=1, keepdims=True)
    amax = np.abs(phi).max(axis=1) + np.abs(mu[:, 0])
    assert np.all(np.abs(phi - mu).max(axis=1) <= amax)
    c = scale_of(amax.max(), 11)
    assert np.abs(c * (phi - mu)).max() < 2.0 ** 12
    hi, lo = split16(c * (phi - mu))
    assert np.abs(hi).max() < 65504 and np.all(np.isfinite(lo))
