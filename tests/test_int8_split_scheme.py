"""The arithmetic behind the INT8 tensor-pipe products of the Rayleigh-Ritz (csrc/rr_i8.cu), restated
in numpy integers and checked on the CPU: the digit split is exact, the bias trick gives the balanced digits, INT32
accumulation cannot overflow at the stated sizes, and the 28 kept digit pairs reproduce a dot product to a few FP64 ulps
of (max of one vector) x (max of the other).  Pins the scheme, not the CUDA code (tests/test_gpu_rr_i8.py does that)."""
import numpy as np

S = 7                       # digit planes per operand
BIAS = 0x0080808080808080   # 128 in each of the 7 low bytes


def fixed_point(x):
    """(q, e): q = rint(x 2^(54 - e)) with |x| 2^-e < 1 for the largest entry (one scale per vector)."""
    mx = np.abs(x).max()
    e = int(np.floor(np.log2(mx))) + 1 if mx > 0 else 0
    q = np.rint(np.ldexp(x, 54 - e)).astype(np.int64)
    return q, e


def digits_loop(q):
    """balanced base-256 digits, least significant first, the schoolbook way"""
    q = q.copy()
    out = []
    for _ in range(S):
        d = ((q & 0xFF) ^ 0x80) - 0x80          # low byte as a signed int8
        out.append(d)
        q = (q - d) >> 8
    assert np.all(q == 0)
    return out


def digits_bias(q):
    """the kernels' way: byte k of q + BIAS with its top bit flipped, read as an int8 (= that byte minus 128)"""
    b = (q + BIAS).astype(np.uint64)
    flipped = [(((b >> np.uint64(8 * k)) & np.uint64(0xFF)).astype(np.int64)) ^ 0x80 for k in range(S)]
    return [(v ^ 0x80) - 0x80 for v in flipped]          # two's-complement reading of the 8-bit pattern


def test_digits_are_exact_balanced_and_the_bias_trick_gives_them():
    rng = np.random.default_rng(0)
    x = rng.standard_normal(4096) * 10.0 ** rng.uniform(-14, 0, 4096)
    x[:4] = [x.max() * 0 + 1.0 - 2.0 ** -53, -(1.0 - 2.0 ** -53), 0.0, 2.0 ** -60]   # edge values under a maximum near 1
    x[4] = 1.0
    q, e = fixed_point(x)
    assert np.abs(q).max() <= 2 ** 54
    dl, db = digits_loop(q), digits_bias(q)
    for a, b in zip(dl, db):
        assert np.array_equal(a, b)
        assert a.min() >= -128 and a.max() <= 127
    recon = sum(d.astype(object) * 256 ** k for k, d in enumerate(dl))
    assert np.all(recon == q.astype(object))
    # the largest entry keeps all 53 mantissa bits; every entry is within 2^-55 of the vector maximum's scale
    err = np.abs(np.ldexp(q.astype(np.float64), e - 54) - x)
    assert err.max() <= 2.0 ** (e - 55)
    big = np.abs(x) >= 2.0 ** (e - 1)
    assert np.all(err[big] == 0.0)


def test_int32_accumulators_cannot_overflow_at_the_stated_sizes():
    # one anti-diagonal d holds d + 1 <= 7 digit pairs of magnitude <= 2^14, K terms each
    assert 7 * 16384 * 128 * 128 < 2 ** 31          # rotation: K = N <= 16384; Gram: 128 K blocks of 128 rows per flush
    assert not (7 * 18725 * 128 * 128 < 2 ** 31)     # the bound is tight to within a few per cent


def test_the_28_kept_digit_pairs_reproduce_a_dot_product_to_a_few_ulps():
    rng = np.random.default_rng(1)
    worst = 0.0
    for K in (16, 260, 2400):
        for _ in range(20):
            y = rng.standard_normal(K) * 10.0 ** rng.uniform(-12, 0, K)
            z = rng.standard_normal(K) * 10.0 ** rng.uniform(-3, 0, K)
            qy, ey = fixed_point(y)
            qz, ez = fixed_point(z)
            dy = digits_loop(qy)[::-1]               # most significant first, like the planes
            dz = digits_loop(qz)[::-1]
            acc = [0] * S                            # one exact integer accumulator per anti-diagonal s + t
            for s in range(S):
                for t in range(S - s):
                    v = int(np.dot(dy[s], dz[t]))
                    assert abs(v) < 2 ** 31 or K > 16384
                    acc[s + t] += v
            val = sum(np.longdouble(a) * np.longdouble(2.0) ** (-8 * d) for d, a in enumerate(acc))
            got = float(val * np.longdouble(2.0) ** (ey + ez - 12))
            ref = float(np.dot(y.astype(np.longdouble), z.astype(np.longdouble)))
            scale = np.abs(y).max() * np.abs(z).max()
            ulps = abs(got - ref) / scale * 2.0 ** 53
            worst = max(worst, ulps / np.sqrt(K))
            assert ulps <= 8.0 * np.sqrt(K), (K, ulps)
    assert worst > 0.0                               # the truncation is visible, just small
