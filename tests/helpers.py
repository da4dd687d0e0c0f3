"""Independent brute-force helpers for pinning the oracle (pure numpy / python).

Nothing here is shared with oracle/ or with the CUDA path: these restate the
*definitions* (Sec. 3-5) in the most literal way, for tiny inputs.
"""
import numpy as np

L = 21
KEY_END = 1 << 63


def decode_key(k):
    """key -> (gx, gy, gz): digit i (from the top) = 4*xbit + 2*ybit + zbit (A3)."""
    k = int(k)
    gx = gy = gz = 0
    for i in range(L):                      # i-th octal digit from the most significant
        digit = (k >> (3 * (L - 1 - i))) & 7
        gx = (gx << 1) | ((digit >> 2) & 1)
        gy = (gy << 1) | ((digit >> 1) & 1)
        gz = (gz << 1) | (digit & 1)
    return gx, gy, gz


def leaf_level(delta):
    """delta = 8^m  ->  L - m; raises if delta is not a power of 8 (Eq. 2)."""
    delta = int(delta)
    m = 0
    while delta > 1:
        assert delta % 8 == 0, "gap is not a power of 8"
        delta //= 8
        m += 1
    assert delta == 1
    return L - m


def check_cornerstone(K):
    """Eq. 2 + alignment: returns the leaf levels."""
    K = [int(v) for v in K]
    assert K[0] == 0 and K[-1] == KEY_END
    levels = []
    for a, b in zip(K[:-1], K[1:]):
        assert b > a
        lv = leaf_level(b - a)
        assert a % (b - a) == 0, "leaf start not divisible by its length"
        levels.append(lv)
    return levels


def random_octree(rng, max_leaves=300, max_level=8, p_split=0.5):
    """A random valid cornerstone array (python ints), by random top-down splitting."""
    leaves = [(0, 0)]  # (start, level)
    changed = True
    while changed and len(leaves) < max_leaves:
        changed = False
        out = []
        for (s, lv) in leaves:
            if lv < max_level and len(out) + 8 < max_leaves and rng.random() < p_split:
                d = 8 ** (L - lv - 1)
                out.extend((s + c * d, lv + 1) for c in range(8))
                changed = True
            else:
                out.append((s, lv))
        leaves = out
        p_split *= 0.8
    return np.array([s for s, _ in leaves] + [KEY_END], dtype=np.uint64)


def grid_coords(c, lo, hi):
    """Integer grid coordinates for a power-of-two-friendly box, in exact arithmetic
    (python fractions), used only where the quotient is exactly representable."""
    from fractions import Fraction
    out = []
    for v in c:
        t = (Fraction(float(v)) - Fraction(float(lo))) / (Fraction(float(hi)) - Fraction(float(lo)))
        g = int(t * (1 << L) // 1)
        out.append(min(max(g, 0), (1 << L) - 1))
    return out
