"""Independent fp64 brute force used ONLY to pin the oracle (tests, `-m "not gpu"`).

Written from the definitions, sharing nothing with oracle/ or the CUDA path: numpy einsum / python
``sorted`` / integer bit manipulation.  Small inputs only.
"""
import numpy as np


def bits_to_f64(u16):
    u16 = np.asarray(u16, dtype=np.uint16)
    return (u16.astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def f64_to_bf16_bits(x):
    """Round-to-nearest-even float64 -> bf16 by integer arithmetic on the float64 bit pattern.
    Valid for finite values whose magnitude is 0 or inside the bf16 normal range (tests stay there)."""
    x = np.asarray(x, dtype=np.float64)
    b = x.view(np.uint64)
    sign = (b >> np.uint64(63)).astype(np.uint32)
    exp = ((b >> np.uint64(52)) & np.uint64(0x7FF)).astype(np.int64)
    man = b & np.uint64((1 << 52) - 1)
    drop = np.uint64(45)  # 52 - 7 mantissa bits kept
    keep = (man >> drop).astype(np.int64)
    rem = man & np.uint64((1 << 45) - 1)
    half = np.uint64(1 << 44)
    round_up = (rem > half) | ((rem == half) & ((keep & 1) == 1))
    keep = keep + round_up.astype(np.int64)
    carry = keep >> 7
    keep = keep & 0x7F
    e = exp - 1023 + 127 + carry
    zero = (exp == 0)
    assert np.all(zero | ((e > 0) & (e < 255))), "outside bf16 normal range"
    out = (sign << 15) | (np.where(zero, 0, e).astype(np.uint32) << 7) | np.where(zero, 0, keep).astype(np.uint32)
    return out.astype(np.uint16)


def pool(kv_bits):
    """Mean over the S keys of each block (Eq.2 with kernel = stride = S)."""
    k = bits_to_f64(kv_bits[:, :, 0])          # [R][Nb][S][D]
    return f64_to_bf16_bits(k.sum(axis=2) / k.shape[2])


def score(F_bits, kpool_bits):
    return np.einsum("rd,rjd->rj", bits_to_f64(F_bits), bits_to_f64(kpool_bits))


def topk_rows(scores_f32, k, n_cand=None):
    """Exhaustive: python sort on (score desc, index asc); ascending ids, -1 padded."""
    scores_f32 = np.asarray(scores_f32, dtype=np.float32)
    R, Nb = scores_f32.shape
    n_cand = Nb if n_cand is None else n_cand
    out = np.full((R, k), -1, dtype=np.int32)
    for r in range(R):
        order = sorted(range(n_cand), key=lambda j: (-float(scores_f32[r, j]), j))
        sel = sorted(order[:k])
        out[r, :len(sel)] = sel
    return out


def attn_over_blocks(Q_bits, kv_bits, ids):
    """Softmax attention of every query head over the tokens of the listed blocks of the FULL cache
    kv [R][Nb][2][S][D]; fp64 throughout.  Returns float64 [B][Hq][D]."""
    Q = bits_to_f64(Q_bits)
    kv = bits_to_f64(kv_bits)
    B, Hq, D = Q.shape
    R = kv.shape[0]
    Hkv = R // B
    G = Hq // Hkv
    O = np.zeros((B, Hq, D))
    for b in range(B):
        for h in range(Hq):
            r = b * Hkv + h // G
            sel = [j for j in ids[r] if j >= 0]
            if not sel:
                continue
            K = kv[r, sel, 0].reshape(-1, D)
            V = kv[r, sel, 1].reshape(-1, D)
            z = K @ Q[b, h] / np.sqrt(D)
            p = np.exp(z - z.max())
            p /= p.sum()
            O[b, h] = p @ V
    return O
