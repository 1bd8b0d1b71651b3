"""Parity rules of BASELINE.json's north_star, shared by the `-m gpu` tests.

ids:       set-equal per row, or every id in the symmetric difference has an oracle score within
           1e-3 * max(|s_(k)|, |s_(k+1)|) of the oracle's k-th score (near-tie band).
gather:    byte-exact.
attention: max-abs <= 2e-2 and mean-abs <= 2e-3 on bf16 outputs compared as floats.
"""
import numpy as np

ATTN_MAX_ABS = 2e-2
ATTN_MEAN_ABS = 2e-3
BAND_REL = 1e-3
# (rows checked, rows that needed the near-tie band) per check_ids call; tests/conftest.py prints the totals per test
BAND_LOG = []


def bits_to_f32(u16):
    return (np.asarray(u16, dtype=np.uint16).astype(np.uint32) << 16).view(np.float32)


def check_ids(gpu_ids, oracle_ids, oracle_scores, n_cand=None):
    """Returns the number of rows that needed the near-tie band; raises AssertionError on a real mismatch.
    gpu_ids / oracle_ids [R][k] int32, oracle_scores [R][Nb] fp32."""
    gpu_ids = np.asarray(gpu_ids)
    oracle_ids = np.asarray(oracle_ids)
    R, k = oracle_ids.shape
    assert gpu_ids.shape == oracle_ids.shape, (gpu_ids.shape, oracle_ids.shape)
    band_rows = 0
    for r in range(R):
        g, o = gpu_ids[r], oracle_ids[r]
        gv = g[g >= 0]
        assert np.all(np.diff(gv) > 0), f"row {r}: ids not strictly ascending: {g}"
        n_valid = int((o >= 0).sum())
        assert len(gv) == n_valid and np.all(g[n_valid:] == -1), f"row {r}: wrong count / padding: {g} vs {o}"
        nc = oracle_scores.shape[1] if n_cand is None else (n_cand if np.isscalar(n_cand) else n_cand[r])
        assert np.all(gv < nc), f"row {r}: id outside the candidate range"
        if np.array_equal(g, o):
            continue
        s = oracle_scores[r, :nc].astype(np.float64)
        srt = np.sort(s)[::-1]
        sk, sk1 = srt[n_valid - 1], srt[n_valid] if n_valid < nc else srt[n_valid - 1]
        tol = BAND_REL * max(abs(sk), abs(sk1))
        diff = np.setxor1d(gv, o[o >= 0])
        assert np.all(np.abs(s[diff] - sk) <= tol), (
            f"row {r}: ids differ outside the near-tie band: gpu-only {np.setdiff1d(gv, o)}, "
            f"oracle-only {np.setdiff1d(o, gv)}, scores {s[diff]}, s_k {sk}, tol {tol}")
        band_rows += 1
    BAND_LOG.append((R, band_rows))
    return band_rows


def check_attn(gpu_O_bits, oracle_O_bits, what=""):
    g = bits_to_f32(gpu_O_bits).astype(np.float64)
    o = bits_to_f32(oracle_O_bits).astype(np.float64)
    assert g.shape == o.shape
    assert np.all(np.isfinite(g)), f"{what}: non-finite attention output"
    d = np.abs(g - o)
    assert d.max() <= ATTN_MAX_ABS, f"{what}: max-abs {d.max():.4g} > {ATTN_MAX_ABS}"
    assert d.mean() <= ATTN_MEAN_ABS, f"{what}: mean-abs {d.mean():.4g} > {ATTN_MEAN_ABS}"
    return float(d.max()), float(d.mean())


def ulp_diff_bf16(a_bits, b_bits):
    """Distance in bf16 ulps between two bit patterns of the same sign (sign-magnitude -> ordered ints)."""
    def key(u):
        u = np.asarray(u, dtype=np.uint16).astype(np.int32)
        return np.where(u & 0x8000, -(u & 0x7FFF), u & 0x7FFF)
    return np.abs(key(a_bits) - key(b_bits))
