"""Host-side model of the routed permutation (csrc/kernels.cuh: pass A native -> coarse buckets, pass B -> caller tiles,
pass C inside the tile; index arrays from four stable sorts, purify_op.cu build_bins_x).  The CUDA path is checked
bit-exactly against purify_op_permutation on the GPU (tests/test_gpu_parity.py::test_routed_permutation_is_the_permutation);
this numpy restatement of the SAME construction, at scaled-down block / tile / bucket sizes, pins the algorithm itself:
ragged last block, last bucket and last tile, padding slots anywhere, blocks that straddle two buckets, and the bit
budgets of the sort keys at the largest supported sizes."""
import numpy as np
import pytest

NONE = 0xFFFFFFFF


def build(perm, M, ts, bs, cs):
    """Index arrays exactly as the create-time kernels compute them (tile = 2^ts, block = 2^bs, bucket = 2^cs elements)."""
    S = len(perm)
    real = perm != NONE
    n_tiles = (M + (1 << ts) - 1) >> ts
    slots = np.arange(S)
    # (1) mid order: stable sort by caller tile, padding last
    key = np.where(real, perm >> ts, n_tiles)
    slot_of_mid = slots[np.argsort(key, kind="stable")][:M]
    q = np.full(S, NONE, dtype=np.int64)
    q[slot_of_mid] = np.arange(M)
    loc_c = perm[slot_of_mid] & ((1 << ts) - 1)
    # (2) A order: stable sort by coarse bucket
    g = np.where(real, perm >> cs, 511)
    slot_a = slots[np.argsort(g, kind="stable")][:M]
    apos = np.full(S, NONE, dtype=np.int64)
    apos[slot_a] = np.arange(M)
    # (3) pass A: order inside every native block by bucket
    order1 = slots[np.argsort(((slots >> bs) << 9) | g, kind="stable")]
    loc_a = np.full(S, 0xFFFF, dtype=np.int64)
    dst_a = np.full(S, NONE, dtype=np.int64)
    p = np.arange(S)
    r1 = real[order1]
    loc_a[order1[r1]] = p[r1] & ((1 << bs) - 1)
    dst_a[p[r1]] = apos[order1[r1]]
    # (4) pass B: order inside every A block by tile (relative to the bucket the block starts in)
    k = np.arange(M)
    kb = cs - ts + 1
    blk = k >> bs
    tile = perm[slot_a] >> ts
    g0 = perm[slot_a[blk << bs]] >> cs
    rel = tile - (g0 << (cs - ts))
    assert (rel >= 0).all() and (rel < (1 << kb)).all()          # the key's bit budget
    order2 = k[np.argsort((blk << kb) | rel, kind="stable")]
    loc_b = np.empty(M, dtype=np.int64)
    loc_b[order2] = np.arange(M) & ((1 << bs) - 1)
    dst_b = q[slot_a[order2]]
    return loc_a, dst_a, loc_b, dst_b, loc_c


def route(src, loc, dst, n_far, bs, inverse=False, far=None):
    """One routing pass over blocks of 2^bs elements (route_kernel, DIR 0 / DIR 1)."""
    B = 1 << bs
    n = len(loc)
    if not inverse:
        out = np.full(n_far, np.nan + 0j)
        for base in range(0, n, B):
            m = min(B, n - base)
            sh = np.full(B, np.nan + 0j)
            l = loc[base:base + m]
            ok = l != 0xFFFF
            sh[l[ok]] = src[base:base + m][ok]
            d = dst[base:base + m]
            okd = d != NONE
            out[d[okd]] = sh[:m][okd]
        return out
    out = np.zeros(n, dtype=complex)
    for base in range(0, n, B):
        m = min(B, n - base)
        sh = np.full(B, np.nan + 0j)
        d = dst[base:base + m]
        okd = d != NONE
        sh[:m][okd] = far[d[okd]]
        l = loc[base:base + m]
        ok = l != 0xFFFF
        blk = np.zeros(m, dtype=complex)
        blk[ok] = sh[l[ok]]
        out[base:base + m] = blk
    return out


def tile_permute(v, loc_c, ts, inverse=False):
    T = 1 << ts
    out = np.empty_like(v)
    for base in range(0, len(v), T):
        m = min(T, len(v) - base)
        l = loc_c[base:base + m]
        if not inverse:
            t = np.full(m, np.nan + 0j)
            t[l] = v[base:base + m]
            out[base:base + m] = t
        else:
            out[base:base + m] = v[base:base + m][l]
    return out


@pytest.mark.parametrize("M,pad,ts,bs,cs", [(1000, 77, 3, 5, 6), (4096, 0, 4, 6, 7), (5003, 1200, 4, 6, 8), (777, 5, 3, 5, 6),
                                            (2048 + 1, 300, 4, 5, 7)])
def test_three_passes_compose_to_the_permutation(M, pad, ts, bs, cs):
    assert cs >= ts + 3 and (1 << cs) >= (1 << bs)               # a block never covers more than two buckets
    rng = np.random.default_rng(M + pad)
    S = M + pad
    perm = np.full(S, NONE, dtype=np.int64)
    perm[rng.permutation(S)[:M]] = rng.permutation(M)
    loc_a, dst_a, loc_b, dst_b, loc_c = build(perm, M, ts, bs, cs)
    real = perm != NONE
    # native -> caller
    v_nat = rng.normal(size=S) + 1j * rng.normal(size=S)
    a = route(v_nat, loc_a, dst_a, M, bs)
    mid = route(a, loc_b, dst_b, M, bs)
    out = tile_permute(mid, loc_c, ts)
    ref = np.empty(M, dtype=complex)
    ref[perm[real]] = v_nat[real]
    assert np.array_equal(out, ref)
    # caller -> native (padding slots 0)
    v_call = rng.normal(size=M) + 1j * rng.normal(size=M)
    mid2 = tile_permute(v_call, loc_c, ts, inverse=True)
    a2 = route(None, loc_b, dst_b, M, bs, inverse=True, far=mid2)
    nat2 = route(None, loc_a, dst_a, M, bs, inverse=True, far=a2)
    ref2 = np.zeros(S, dtype=complex)
    ref2[real] = v_call[perm[real]]
    assert np.array_equal(nat2, ref2)
    # runs: consecutive sorted ranks of one block that share a bucket (pass A) go to consecutive destinations
    d = dst_a[:(S >> bs) << bs].reshape(-1, 1 << bs)
    both = (d[:, 1:] != NONE) & (d[:, :-1] != NONE)
    breaks = both & (np.diff(d, axis=1) != 1)
    n_buckets = ((M - 1) >> cs) + 1
    assert breaks.sum(axis=1).max() <= n_buckets - 1


@pytest.mark.parametrize("M,complex128", [(1 << 24, False), (10 ** 8, False), (5 * 10 ** 8, False), ((1 << 31) - 1, False),
                                          ((1 << 31) - 1, True)])
def test_sort_key_bit_budgets(M, complex128):
    """The four radix sorts use 32-bit keys: bucket count <= 256 (9 bits with the padding code), block and tile fields fit."""
    ts, bs = 12, 12 if complex128 else 13
    cs = ts + 3
    while ((M - 1) >> cs) >= 256:
        cs += 1
    S = int(M * 1.25)                                           # generous padding ratio
    nbits = lambda v: max(1, int(v).bit_length())
    assert ((M - 1) >> cs) < 256 and (1 << cs) >= (1 << bs)
    assert 9 + nbits((S - 1) >> bs) <= 32                        # sort (3)
    assert (cs - ts + 1) + nbits((M - 1) >> bs) <= 32            # sort (4)
    assert nbits((M + (1 << ts) - 1) >> ts) <= 32                # sort (1)
