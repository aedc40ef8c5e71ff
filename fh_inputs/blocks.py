"""Seeded random block entries and block-key enumeration (no method arithmetic)."""
import numpy as np

from .profiles import SITE_LABELS, fuse_labels

# (q, 2k) of the MPO bond multiplets S, P, M, F (reduced MPO bond dimension 4)
MPO_LABELS = ((0, 0), (1, 1), (-1, 1), (0, 0))


def site_block_keys(dims_l, dims_r):
    """Keys (a, s, c) of a one-site tensor between bonds with profiles dims_l, dims_r."""
    keys = []
    for a in sorted(dims_l):
        for s in range(3):
            for c in fuse_labels(a, s):
                if c in dims_r:
                    keys.append((a, s, c))
    return sorted(keys)


def theta_block_keys(dims_l, dims_r):
    """Keys (a, s1, c, s2, b) of a two-site tensor; c is any label allowed by fusion."""
    keys = []
    for a in sorted(dims_l):
        for s1 in range(3):
            for c in fuse_labels(a, s1):
                for s2 in range(3):
                    for b in fuse_labels(c, s2):
                        if b in dims_r:
                            keys.append((a, s1, c, s2, b))
    return sorted(keys)


def env_block_keys(dims_bra, dims_ket):
    """Keys (x', w, x) of an environment: q_x' = q_x + q_w, |j_x - k_w| <= j_x' <= j_x + k_w."""
    keys = []
    for xp in sorted(dims_bra):
        for w in range(4):
            qw, tk = MPO_LABELS[w]
            for x in sorted(dims_ket):
                if xp[0] == x[0] + qw and abs(x[1] - tk) <= xp[1] <= x[1] + tk \
                        and (x[1] + tk + xp[1]) % 2 == 0:
                    keys.append((xp, w, x))
    return sorted(keys)


def _flatten(key):
    out = []
    for part in key:
        if isinstance(part, tuple):
            out.extend(part)
        else:
            out.append(part)
    return out


def _counter_words(key):
    """Pack the integer labels of a block key into three uint64 words (one byte per label,
    offset by 128)."""
    labels = _flatten(key)
    assert len(labels) <= 24
    words = [0, 0, 0]
    if all(-128 <= int(v) < 128 for v in labels):
        for i, v in enumerate(labels):
            words[i // 8] |= (int(v) + 128) << (8 * (i % 8))
        return words
    # wide labels (the packed charges of the U(1) x U(1) mode): two bytes per label, top bit of the last word set
    assert len(labels) <= 11
    for i, v in enumerate(labels):
        b = int(v) + 32768
        assert 0 <= b < 65536
        words[i // 4] |= b << (16 * (i % 4))
    words[2] |= 1 << 63
    return words


def random_blocks(seed, tag, keys, shapes, scale=None):
    """{key: complex128 array} with iid entries N(0,1) + i N(0,1) (optionally * scale[key]).

    Counter-based: block `key` of tensor `tag` always gets the same numbers, whatever other
    blocks are generated -- Philox with key (seed, tag) and the 256-bit counter's upper three
    words holding the block's labels.
    """
    out = {}
    for key in keys:
        w = _counter_words(key)
        bg = np.random.Philox(key=[int(seed), int(tag)], counter=[0, w[0], w[1], w[2]])
        g = np.random.Generator(bg)
        m, n = shapes[key]
        z = g.standard_normal((m, n, 2))
        blk = z[..., 0] + 1j * z[..., 1]
        if scale is not None:
            blk = blk * scale[key]
        out[key] = np.ascontiguousarray(blk)
    return out
