"""Pins for the CPU oracle (SURVEY.md §8(c) "What pins each part").

The paper prints no worked numeric example for this path, so every oracle function is pinned by
an independent fp64 brute force (tests/bruteforce.py), by invariants the paper fixes, by special
cases with closed forms and by reduction to a library routine.  All CPU, `-m "not gpu"`.
"""
import math
import os

import numpy as np
import pytest
import torch

from paper_2606_04511_b200 import synth
import bruteforce as bf

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _layer(cfg, layer=0):
    from oracle import sparda_oracle as o
    d = synth.decode_layer(cfg, layer, device="cpu")
    return {k: o.from_torch(v) for k, v in d.items()}


SMALL = synth.DecodeConfig("small", batch=2, n_q_heads=8, n_kv_heads=2, head_dim=64, n_blocks=12, topk=5,
                           bias_std=1.5, seed=11)


# ---------------------------------------------------------------- bf16 rounding
def test_bf16_rounding_matches_torch_and_bit_arithmetic(oracle):
    rng = np.random.default_rng(0)
    x32 = np.concatenate([
        rng.standard_normal(4000).astype(np.float32) * np.float32(10.0) ** rng.integers(-20, 20, 4000).astype(np.float32),
        np.array([0.0, -0.0, 1.0, -1.0, 1.0 + 2.0 ** -8, 1.0 + 3 * 2.0 ** -8, 1.0 + 2.0 ** -8 + 2.0 ** -20,
                  255.5, 256.5, 3.3895314e38, 1e-38, 1.1754944e-38, 9.2e-41, 4.6e-41], dtype=np.float32)])
    want = torch.from_numpy(x32).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    got = np.array([oracle.double_to_bf16(float(v)) for v in x32], dtype=np.uint16)
    np.testing.assert_array_equal(got, want)
    # exact ties in double (not representable in fp32 paths): 1 + 2^-8 is a tie -> even (1.0); just above -> up
    assert oracle.double_to_bf16(1.0 + 2.0 ** -8) == 0x3F80
    assert oracle.double_to_bf16(1.0 + 2.0 ** -8 + 2.0 ** -40) == 0x3F81
    assert oracle.double_to_bf16(1.0 + 3 * 2.0 ** -8) == 0x3F82
    assert oracle.double_to_bf16(float("inf")) == 0x7F80 and oracle.double_to_bf16(-float("inf")) == 0xFF80
    assert oracle.double_to_bf16(1e39) == 0x7F80
    # the independent integer-arithmetic rounding agrees on normal-range doubles
    xd = rng.standard_normal(2000) * 7.0
    np.testing.assert_array_equal(np.array([oracle.double_to_bf16(float(v)) for v in xd], dtype=np.uint16),
                                  bf.f64_to_bf16_bits(xd))
    # widening is exact
    bits = rng.integers(0, 0x7F80, 1000).astype(np.uint16)
    np.testing.assert_array_equal(oracle.bf16_bits_to_f64(bits), bf.bits_to_f64(bits))


# ---------------------------------------------------------------- o1 pooling (Eq.2)
def test_pool_matches_bruteforce_and_constant_block(oracle):
    L = _layer(SMALL)
    kp = oracle.pool_keys(L["kv"])
    np.testing.assert_array_equal(kp, bf.pool(L["kv"]))
    kv = L["kv"].copy()
    c = oracle.double_to_bf16(-2.75)
    kv[0, 3, 0] = c
    assert np.all(oracle.pool_keys(kv)[0, 3] == c)
    # V plane must not leak into the pooled keys
    kv2 = L["kv"].copy()
    kv2[:, :, 1] = 0
    np.testing.assert_array_equal(oracle.pool_keys(kv2), kp)


def test_pool_linearity_bound(oracle):
    """F . mean(K) = mean_t(F . k_t) up to the single bf16 rounding of Kpool (bound 2^-8 sum|F_d Kp_d|)."""
    L = _layer(SMALL)
    kp = oracle.pool_keys(L["kv"])
    s = oracle.score(L["F"], kp).astype(np.float64)
    F = bf.bits_to_f64(L["F"])
    K = bf.bits_to_f64(L["kv"][:, :, 0])
    token_level = np.einsum("rd,rjtd->rjt", F, K).mean(axis=2)
    bound = 2.0 ** -8 * np.einsum("rd,rjd->rj", np.abs(F), np.abs(bf.bits_to_f64(kp))) + 1e-5
    assert np.all(np.abs(s - token_level) <= bound)


# ---------------------------------------------------------------- o3 + o4 selection (Eq.4)
def test_score_matches_bruteforce(oracle):
    L = _layer(SMALL)
    kp = oracle.pool_keys(L["kv"])
    np.testing.assert_array_equal(oracle.score(L["F"], kp), bf.score(L["F"], kp).astype(np.float32))


@pytest.mark.parametrize("seed", range(6))
def test_topk_exhaustive_tiny(oracle, seed):
    """(i1) exhaustive python sort on tiny inputs, incl. heavy ties and k > n_cand."""
    rng = np.random.default_rng(seed)
    R, Nb = 5, int(rng.integers(1, 17))
    k = int(rng.integers(1, Nb + 3))
    s = rng.integers(-3, 4, size=(R, Nb)).astype(np.float32) if seed % 2 else rng.standard_normal((R, Nb)).astype(np.float32)
    n_cand = int(rng.integers(0, Nb + 1))
    np.testing.assert_array_equal(oracle.topk(s, k), bf.topk_rows(s, k))
    np.testing.assert_array_equal(oracle.topk(s, k, n_cand), bf.topk_rows(s, k, n_cand))


def test_select_cfg1_exhaustive(oracle):
    L = _layer(synth.CFG1_TINY)
    kp = oracle.pool_keys(L["kv"])
    ids, s = oracle.forecast_select(L["F"], kp, synth.CFG1_TINY.topk)
    np.testing.assert_array_equal(ids, bf.topk_rows(bf.score(L["F"], kp).astype(np.float32), synth.CFG1_TINY.topk))
    assert ids.shape == (1, 8) and np.all(np.diff(ids, axis=1) > 0)


def test_no_softmax_invariant(oracle):
    """(i2) P:L91: ranking raw Forecast logits == ranking their softmax == ranking any positive multiple."""
    rng = np.random.default_rng(3)
    R, Nb, k = 4, 64, 8
    raw = np.stack([rng.permutation(Nb) for _ in range(R)]).astype(np.float32) * 0.25 - 7.0  # gaps of 0.25
    sm = np.exp(raw.astype(np.float64) - raw.max(axis=1, keepdims=True))
    sm = (sm / sm.sum(axis=1, keepdims=True)).astype(np.float32)
    base = oracle.topk(raw, k)
    np.testing.assert_array_equal(oracle.topk(sm, k), base)
    np.testing.assert_array_equal(oracle.topk(raw * np.float32(3.5), k), base)
    np.testing.assert_array_equal(base, np.sort(np.argsort(-raw, axis=1)[:, :k], axis=1).astype(np.int32))


def test_topk_structural_invariants(oracle):
    rng = np.random.default_rng(4)
    R, Nb, k = 3, 40, 7
    s = rng.standard_normal((R, Nb)).astype(np.float32)
    # (i3) k = Nb returns every block
    np.testing.assert_array_equal(oracle.topk(s, Nb), np.tile(np.arange(Nb, dtype=np.int32), (R, 1)))
    # (i4) permuting blocks permutes the ids
    perm = rng.permutation(Nb)
    ids = oracle.topk(s, k)
    ids_p = oracle.topk(s[:, perm], k)
    for r in range(R):
        assert set(perm[ids_p[r]]) == set(ids[r])
    # (i6) all-equal scores -> lowest indices
    np.testing.assert_array_equal(oracle.topk(np.zeros((2, Nb), np.float32), k), np.tile(np.arange(k, dtype=np.int32), (2, 1)))
    # (i7) a duplicated block: the lower index is taken first
    s2 = np.full((1, Nb), -5.0, np.float32)
    s2[0, [9, 30]] = 2.0
    np.testing.assert_array_equal(oracle.topk(s2, 1), [[9]])
    # fewer candidates than k: all candidates then -1 (q5); zero candidates: all -1
    np.testing.assert_array_equal(oracle.topk(s, k, 3), np.tile(np.array([0, 1, 2, -1, -1, -1, -1], np.int32), (R, 1)))
    assert np.all(oracle.topk(s, k, 0) == -1)
    # -inf and +inf scores order correctly
    s3 = np.array([[0.0, -np.inf, np.inf, 1.0, -1.0]], np.float32)
    np.testing.assert_array_equal(oracle.topk(s3, 2), [[2, 3]])
    np.testing.assert_array_equal(oracle.topk(s3, 4), [[0, 2, 3, 4]])


def test_planted_needle_is_selected(oracle):
    """(i5) a block whose pooled key is a large multiple of F must be selected."""
    L = _layer(SMALL)
    kp = oracle.pool_keys(L["kv"])
    F = bf.bits_to_f64(L["F"])
    kp2 = kp.copy()
    for r in range(kp.shape[0]):
        kp2[r, 7] = bf.f64_to_bf16_bits(8.0 * F[r])
    ids, _ = oracle.forecast_select(L["F"], kp2, 1)
    assert np.all(ids[:, 0] == 7)


# ---------------------------------------------------------------- o5 gather
def test_gather_exact_bytes_and_untouched_slots(oracle):
    L = _layer(SMALL)
    R, Nb = L["kv"].shape[:2]
    rng = np.random.default_rng(5)
    k = 6
    ids = np.stack([np.sort(rng.choice(Nb, k, replace=False)) for _ in range(R)]).astype(np.int32)
    ids[1, 4:] = -1
    pool = np.full((R, k, 2, SMALL.block_size, SMALL.head_dim), 0xABCD, dtype=np.uint16)
    oracle.gather(L["kv"], ids, pool)
    for r in range(R):
        for i in range(k):
            if ids[r, i] >= 0:
                assert pool[r, i].tobytes() == L["kv"][r, ids[r, i]].tobytes()
            else:
                assert np.all(pool[r, i] == 0xABCD)


# ---------------------------------------------------------------- o6 / o7 attention (Eq.5)
def test_sparse_equals_dense_when_topk_covers_all_blocks(oracle):
    """(j1) k = Nb: sparse attention == dense attention by an independent fp64 brute force."""
    L = _layer(SMALL)
    R, Nb = L["kv"].shape[:2]
    ids = np.tile(np.arange(Nb, dtype=np.int32), (R, 1))
    pool = oracle.gather(L["kv"], ids)
    O, O64 = oracle.sparse_attn(L["Q"], pool, ids)
    Od, Od64 = oracle.dense_attn(L["Q"], L["kv"])
    want = bf.attn_over_blocks(L["Q"], L["kv"], ids)
    np.testing.assert_allclose(O64, want, rtol=0, atol=1e-12)
    np.testing.assert_allclose(Od64, want, rtol=0, atol=1e-12)
    np.testing.assert_array_equal(O, Od)
    np.testing.assert_array_equal(O, bf.f64_to_bf16_bits(np.where(np.abs(want) < 1e-30, 0.0, want)))
    # indexed mode (layer-0 cache) is the same computation
    Oi, Oi64 = oracle.sparse_attn(L["Q"], L["kv"], ids, pool_is_indexed=True)
    np.testing.assert_array_equal(Oi, O)


def test_sparse_attn_matches_bruteforce_and_sdpa(oracle):
    """(j2) reduction to torch.nn.functional.scaled_dot_product_attention over the gathered tokens."""
    L = _layer(SMALL)
    kp = oracle.pool_keys(L["kv"])
    ids, _ = oracle.forecast_select(L["F"], kp, SMALL.topk)
    ids[1, -2:] = -1                                   # a row with padding
    pool = oracle.gather(L["kv"], ids, np.full((SMALL.rows, SMALL.topk, 2, 64, 64), 0x7FC0, np.uint16))  # NaN poison
    O, O64 = oracle.sparse_attn(L["Q"], pool, ids)
    np.testing.assert_allclose(O64, bf.attn_over_blocks(L["Q"], L["kv"], ids), rtol=0, atol=1e-12)
    B, Hq, D, G = SMALL.batch, SMALL.n_q_heads, SMALL.head_dim, SMALL.group
    for r in range(SMALL.rows):
        b, g = divmod(r, SMALL.n_kv_heads)
        sel = [i for i in range(SMALL.topk) if ids[r, i] >= 0]
        K = torch.from_numpy(bf.bits_to_f64(pool[r, sel, 0]).reshape(1, 1, -1, D)).float()
        V = torch.from_numpy(bf.bits_to_f64(pool[r, sel, 1]).reshape(1, 1, -1, D)).float()
        q = torch.from_numpy(bf.bits_to_f64(L["Q"][b, g * G:(g + 1) * G])).float().reshape(1, G, 1, D)
        ref = torch.nn.functional.scaled_dot_product_attention(q, K.expand(1, G, -1, D), V.expand(1, G, -1, D))
        np.testing.assert_allclose(O64[b, g * G:(g + 1) * G], ref.reshape(G, D).double().numpy(), rtol=0, atol=2e-5)


def test_attention_closed_forms(oracle):
    L = _layer(SMALL)
    R, Nb, _, S, D = L["kv"].shape
    k = 4
    ids = np.tile(np.array([1, 4, 6, 9], np.int32), (R, 1))
    # (j3) all V rows = c  =>  O = c (softmax weights sum to one, j7)
    kv = L["kv"].copy()
    c = bf.f64_to_bf16_bits(np.linspace(-2, 2, D))
    kv[:, :, 1] = c
    _, O64 = oracle.sparse_attn(L["Q"], oracle.gather(kv, ids), ids)
    np.testing.assert_allclose(O64, np.broadcast_to(bf.bits_to_f64(c), O64.shape), rtol=0, atol=1e-12)
    # (j4) one selected block with identical keys  =>  O = mean of its V rows
    kv = L["kv"].copy()
    kv[:, 5, 0] = kv[:, 5, 0, :1]
    one = np.full((R, k), -1, np.int32)
    one[:, 0] = 5
    _, O64 = oracle.sparse_attn(L["Q"], oracle.gather(kv, one), one)
    G = SMALL.group
    for b in range(SMALL.batch):
        for h in range(SMALL.n_q_heads):
            r = b * SMALL.n_kv_heads + h // G
            np.testing.assert_allclose(O64[b, h], bf.bits_to_f64(kv[r, 5, 1]).mean(axis=0), rtol=0, atol=1e-12)
    # (j5) adding one vector delta to every key leaves O unchanged (exactly representable shift)
    kv = L["kv"].copy()
    kq = np.round(bf.bits_to_f64(kv[:, :, 0]) * 4) / 4          # quarter-integers, |.| < 16: exact in bf16 after +2
    kq = np.clip(kq, -7.75, 7.75)
    kv[:, :, 0] = bf.f64_to_bf16_bits(kq)
    kv_shift = kv.copy()
    kv_shift[:, :, 0] = bf.f64_to_bf16_bits(kq + 2.0)
    np.testing.assert_array_equal(bf.bits_to_f64(kv_shift[:, :, 0]), kq + 2.0)
    _, Oa = oracle.sparse_attn(L["Q"], oracle.gather(kv, ids), ids)
    _, Ob = oracle.sparse_attn(L["Q"], oracle.gather(kv_shift, ids), ids)
    np.testing.assert_allclose(Oa, Ob, rtol=0, atol=1e-10)
    # (j6) the order of the selected blocks does not matter beyond fp noise
    rev = ids[:, ::-1].copy()
    pool_rev = oracle.gather(L["kv"], rev)
    _, Oc = oracle.sparse_attn(L["Q"], pool_rev, rev)
    _, Od = oracle.sparse_attn(L["Q"], oracle.gather(L["kv"], ids), ids)
    np.testing.assert_allclose(Oc, Od, rtol=0, atol=1e-12)
    # a row with no valid block gives zeros
    none = np.full((R, k), -1, np.int32)
    O, _ = oracle.sparse_attn(L["Q"], oracle.gather(L["kv"], ids), none)
    assert np.all(O == 0)


def test_gqa_head_to_group_mapping(oracle):
    """Query head h reads KV head h // G: zero all but one group's V and see who changes."""
    L = _layer(SMALL)
    R = SMALL.rows
    ids = np.tile(np.array([0, 2, 3], np.int32), (R, 1))
    kv = L["kv"].copy()
    kv[1::2, :, 1] = 0                                  # rows with g = 1
    _, O64 = oracle.sparse_attn(L["Q"], oracle.gather(kv, ids), ids)
    G = SMALL.group
    assert np.all(O64[:, G:] == 0) and np.all(np.abs(O64[:, :G]).sum(axis=-1) > 0)


# ---------------------------------------------------------------- o8 / o9 prefill selection
PRE = synth.PrefillConfig("pre_small", n_q_heads=8, n_kv_heads=2, head_dim=64, seq_len=640, topk=4, chunk=128, seed=7)


def _prefill(cfg):
    from oracle import sparda_oracle as o
    d = synth.prefill_inputs(cfg, "cpu")
    d = {k: o.from_torch(v) for k, v in d.items()}
    d["kpool"] = o.pool_keys(d["kv"])
    return d


def test_prefill_select_rows_equal_decode_selector_on_causal_prefix(oracle):
    P = _prefill(PRE)
    ids, sc = oracle.prefill_select(P["F"], P["kpool"], PRE.topk, want_scores=True)
    assert ids.shape == (2, PRE.seq_len, PRE.topk)
    assert np.all(ids[:, :63] == -1)                                    # q8: rows i < 63 have no candidate
    np.testing.assert_array_equal(ids[:, 63], np.tile(np.array([0, -1, -1, -1], np.int32), (2, 1)))
    for i in [63, 64, 127, 128, 200, 319, 320, 511, 639]:
        n_cand = (i + 1) // 64
        dec_ids, dec_s = oracle.forecast_select(P["F"][:, i], P["kpool"], PRE.topk, n_cand)
        np.testing.assert_array_equal(ids[:, i], dec_ids)
        np.testing.assert_array_equal(sc[:, i, :n_cand], dec_s[:, :n_cand])
        assert np.all(np.isneginf(sc[:, i, n_cand:]))
    # chunked call == slice of the whole
    np.testing.assert_array_equal(oracle.prefill_select(P["F"], P["kpool"], PRE.topk, row0=256, n_rows=128), ids[:, 256:384])


def test_prefill_baseline_bruteforce_and_g1_reduces_to_forecast(oracle):
    P = _prefill(PRE)
    G = PRE.n_q_heads // PRE.n_kv_heads
    ids, sc = oracle.prefill_select_baseline(P["Q"], P["kpool"], PRE.topk, want_scores=True)
    Q = bf.bits_to_f64(P["Q"])
    Kp = bf.bits_to_f64(P["kpool"])
    for g in range(2):
        for i in [63, 130, 400, 639]:
            n = (i + 1) // 64
            z = np.einsum("hd,jd->hj", Q[g * G:(g + 1) * G, i], Kp[g, :n]) / math.sqrt(PRE.head_dim)
            p = np.exp(z - z.max(axis=1, keepdims=True))
            shared = (p / p.sum(axis=1, keepdims=True)).sum(axis=0)
            np.testing.assert_allclose(sc[g, i, :n], shared, rtol=1e-6)
            np.testing.assert_array_equal(ids[g, i], bf.topk_rows(shared[None].astype(np.float32), PRE.topk)[0])
    # G = 1 with Q = F: softmax is monotone, so the baseline selector picks the Forecast selector's blocks
    ids_f = oracle.prefill_select(P["F"], P["kpool"], PRE.topk)
    ids_b = oracle.prefill_select_baseline(P["F"], P["kpool"], PRE.topk)
    np.testing.assert_array_equal(ids_b, ids_f)


# ---------------------------------------------------------------- o10 pipeline wiring
def test_pipeline_wiring_with_planted_needles(oracle):
    cfg = SMALL.with_(n_layers=4, topk=3)
    layers = []
    for l in range(cfg.n_layers):
        L = _layer(cfg, l)
        L["kpool"] = oracle.pool_keys(L["kv"])
        layers.append(L)
    # plant: layer 0 block 2 answers F0cur; layer l>=1 block 3+l answers F_{l-1} (reading q9)
    for r in range(cfg.rows):
        layers[0]["kpool"][r, 2] = bf.f64_to_bf16_bits(8.0 * bf.bits_to_f64(layers[0]["F0cur"][r]))
        for l in range(1, cfg.n_layers):
            layers[l]["kpool"][r, 3 + l] = bf.f64_to_bf16_bits(8.0 * bf.bits_to_f64(layers[l - 1]["F"][r]))
    out = oracle.decode_pipeline(layers, cfg.topk)
    assert all(2 in out[0]["ids"][r] for r in range(cfg.rows))
    for l in range(1, cfg.n_layers):
        assert all(3 + l in out[l]["ids"][r] for r in range(cfg.rows))
    # each layer equals the hand composition, layer 0 reads its own cache by block id (no pool)
    assert out[0]["pool"] is None
    np.testing.assert_allclose(out[0]["O64"], bf.attn_over_blocks(layers[0]["Q"], layers[0]["kv"], out[0]["ids"]), atol=1e-12)
    for l in range(1, cfg.n_layers):
        np.testing.assert_allclose(out[l]["O64"], bf.attn_over_blocks(layers[l]["Q"], layers[l]["kv"], out[l]["ids"]), atol=1e-12)
        for r in range(cfg.rows):
            for i, j in enumerate(out[l]["ids"][r]):
                assert out[l]["pool"][r, i].tobytes() == layers[l]["kv"][r, j].tobytes()


# ---------------------------------------------------------------- o2 Forecast projection (Eq.3; one head per group)
def test_forecast_project_reduces_to_a_matmul(oracle):
    """o2 is a plain GEMV per sequence: it must equal numpy's fp64 matmul rounded once to bf16 (library routine), and
    the column block of group g must depend only on W_F[:, g*D:(g+1)*D] (one Forecast head per KV group)."""
    rng = np.random.default_rng(2)
    B, hidden, Hkv, D = 3, 192, 2, 64
    X = bf.f64_to_bf16_bits(rng.standard_normal((B, hidden)))
    W = bf.f64_to_bf16_bits(rng.standard_normal((hidden, Hkv * D)) / 8)
    F = oracle.forecast_project(X, W, Hkv, D)
    assert F.shape == (B * Hkv, D)
    want = bf.f64_to_bf16_bits(bf.bits_to_f64(X) @ bf.bits_to_f64(W)).reshape(B * Hkv, D)
    assert np.max(parity_ulps(F, want)) <= 1            # the two fp64 sums differ only in order
    W2 = W.copy()
    W2[:, D:] = bf.f64_to_bf16_bits(rng.standard_normal((hidden, D)))
    F2 = oracle.forecast_project(X, W2, Hkv, D)
    np.testing.assert_array_equal(F2.reshape(B, Hkv, D)[:, 0], F.reshape(B, Hkv, D)[:, 0])
    assert not np.array_equal(F2.reshape(B, Hkv, D)[:, 1], F.reshape(B, Hkv, D)[:, 1])


def parity_ulps(a, b):
    def key(u):
        u = np.asarray(u, dtype=np.uint16).astype(np.int32)
        return np.where(u & 0x8000, -(u & 0x7FFF), u & 0x7FFF)
    return np.abs(key(a) - key(b))


# ---------------------------------------------------------------- o11 / o12 block reuse between decode steps
def test_reuse_plan_set_invariants_random(oracle):
    """o11 against what 'only newly selected blocks are fetched' fixes, checked with Python sets written
    here: after the step the pool holds exactly the new selection, re-selected blocks did not move, the fetched
    blocks are exactly new \\ old, nothing else is touched."""
    rng = np.random.default_rng(7)
    for trial in range(200):
        k = int(rng.integers(1, 20))
        nb = int(rng.integers(k, 3 * k + 2))
        R = 3
        old = np.full((R, k), -1, dtype=np.int32)
        new = np.full((R, k), -1, dtype=np.int32)
        for r in range(R):
            m_old = int(rng.integers(0, k + 1))
            m_new = int(rng.integers(0, k + 1))
            old[r, rng.permutation(k)[:m_old]] = rng.permutation(nb)[:m_old]      # unordered slots, some empty
            new[r, :m_new] = np.sort(rng.permutation(nb)[:m_new])                    # ascending, -1 padded
        after, fetch = oracle.reuse_plan(new, old)
        for r in range(R):
            so, sn = set(old[r][old[r] >= 0].tolist()), set(new[r][new[r] >= 0].tolist())
            assert set(after[r][after[r] >= 0].tolist()) == sn
            assert len(after[r][after[r] >= 0]) == len(sn)                           # no duplicates
            assert set(fetch[r][fetch[r] >= 0].tolist()) == sn - so
            for s_ in range(k):
                if old[r, s_] >= 0 and int(old[r, s_]) in sn:
                    assert after[r, s_] == old[r, s_] and fetch[r, s_] == -1          # a hit stays where it is
                if fetch[r, s_] >= 0:
                    assert after[r, s_] == fetch[r, s_]
            # ascending misses meet ascending freed slots
            f = fetch[r][fetch[r] >= 0]
            assert np.all(np.diff(f) > 0)


def test_reuse_plan_special_cases(oracle):
    new = np.array([[2, 5, 9, 11]], dtype=np.int32)
    empty = np.full((1, 4), -1, dtype=np.int32)
    after, fetch = oracle.reuse_plan(new, empty)                 # first step: a plain gather in id order
    np.testing.assert_array_equal(after, new)
    np.testing.assert_array_equal(fetch, new)
    after2, fetch2 = oracle.reuse_plan(new, after)               # same selection again: nothing to fetch
    np.testing.assert_array_equal(after2, after)
    assert np.all(fetch2 == -1)
    after3, fetch3 = oracle.reuse_plan(np.array([[1, 5, 11, 30]], dtype=np.int32), after)
    np.testing.assert_array_equal(after3, [[1, 5, 30, 11]])      # 2 -> 1 (slot 0), 9 -> 30 (slot 2); 5 and 11 stay
    np.testing.assert_array_equal(fetch3, [[1, -1, 30, -1]])
    after4, fetch4 = oracle.reuse_plan(np.array([[5, -1, -1, -1]], dtype=np.int32), after3)
    np.testing.assert_array_equal(after4, [[-1, 5, -1, -1]])     # fewer selected than slots: the rest become empty
    assert np.all(fetch4 == -1)


def test_cached_pipeline_equals_plain_pipeline_step_by_step(oracle):
    """o12: with the block cache the pool holds the same blocks in another slot order, so every step's attention
    equals the cache-free pipeline o10 up to the order of a double-precision sum, the pool slots hold exactly the
    bytes of the blocks slot_ids names, and only new blocks are copied."""
    cfg = SMALL.with_(n_layers=3, topk=4)
    base = []
    for l in range(cfg.n_layers):
        L = _layer(cfg, l)
        L["kpool"] = oracle.pool_keys(L["kv"])
        base.append(L)
    rng = np.random.default_rng(3)
    steps = []
    for t in range(4):
        layers = []
        for l, L in enumerate(base):
            d = dict(L)
            if t > 0:                                             # drift the Forecast a little: selections overlap
                f = bf.bits_to_f64(L["F"]) + 0.6 * t * rng.standard_normal(L["F"].shape)
                d["F"] = bf.f64_to_bf16_bits(f)
            layers.append(d)
        steps.append(layers)
    out, _ = oracle.decode_pipeline_cached(steps, cfg.topk)
    fetched_total = 0
    for t, layers in enumerate(steps):
        plain = oracle.decode_pipeline(layers, cfg.topk)
        for l in range(cfg.n_layers):
            np.testing.assert_array_equal(out[t][l]["ids"], plain[l]["ids"])
            np.testing.assert_allclose(out[t][l]["O64"], plain[l]["O64"], rtol=0, atol=1e-9)
            if l == 0:
                continue
            for r in range(cfg.rows):
                assert sorted(out[t][l]["slot_ids"][r].tolist()) == sorted(plain[l]["ids"][r].tolist())
                for s_, j in enumerate(out[t][l]["slot_ids"][r]):
                    assert out[t][l]["pool"][r, s_].tobytes() == layers[l]["kv"][r, j].tobytes()
            n_f = int((out[t][l]["fetch"] >= 0).sum())
            if t == 0:
                assert n_f == cfg.rows * cfg.topk
            else:
                new_blocks = sum(len(set(out[t][l]["ids"][r].tolist()) - set(out[t - 1][l]["ids"][r].tolist()))
                                 for r in range(cfg.rows))
                assert n_f == new_blocks
                fetched_total += n_f
    assert 0 < fetched_total < 3 * 2 * cfg.rows * cfg.topk       # the drift really produced partial reuse


# ---------------------------------------------------------------- o13 cache maintenance
def test_append_kv_fills_a_block_like_the_prefilled_cache(oracle):
    """Appending a block's 64 tokens one by one to an empty cache must leave exactly the bytes of the prefilled cache and,
    when the block completes, exactly o1's pooled key for it; nothing else changes, and the candidate range grows by one
    block only on completion."""
    cfg = SMALL
    L = _layer(cfg)
    want_kv = L["kv"]
    want_pool = oracle.pool_keys(want_kv)
    R, Nb, _, S, D = want_kv.shape
    kv = np.full_like(want_kv, 0x7FC0)                       # NaN pattern: untouched bytes stay recognisable
    kpool = np.full_like(want_pool, 0x7FC0)
    for t in range(2 * S + 5):                               # two full blocks and a partial third
        j, o = divmod(t, S)
        n = oracle.append_kv(kv, kpool, want_kv[:, j, 0, o], want_kv[:, j, 1, o], t)
        assert n == (t + 1) // S
        if o == S - 1:
            np.testing.assert_array_equal(kpool[:, j], want_pool[:, j])
        else:
            assert np.all(kpool[:, j] == 0x7FC0)             # a partial block has no pooled key yet
    np.testing.assert_array_equal(kv[:, :2], want_kv[:, :2])
    np.testing.assert_array_equal(kv[:, 2, :, :5], want_kv[:, 2, :, :5])
    assert np.all(kv[:, 2, :, 5:] == 0x7FC0) and np.all(kv[:, 3:] == 0x7FC0) and np.all(kpool[:, 2:] == 0x7FC0)


def test_appended_block_becomes_selectable_when_complete(oracle):
    """Planted needle through o13 + o3/o4: a block whose keys all equal 8*F is not a candidate while partial and is
    selected by the first selection after its last token arrives (the index is updated incrementally)."""
    cfg = SMALL.with_(topk=3)
    L = _layer(cfg)
    kv, kpool = L["kv"].copy(), oracle.pool_keys(L["kv"])
    R, Nb, _, S, D = kv.shape
    j = Nb - 1                                               # re-append the last block with needle keys
    needle = bf.f64_to_bf16_bits(8.0 * bf.bits_to_f64(L["F"]))
    for o in range(S):
        n = oracle.append_kv(kv, kpool, needle, L["kv"][:, j, 1, o], j * S + o)
        ids, _ = oracle.forecast_select(L["F"], kpool, cfg.topk, n)
        assert all((j in ids[r]) == (o == S - 1) for r in range(R))


# ---------------------------------------------------------------- o14 / o15 the (32,16) grid + max-pool (reading q19; unpinned by the paper)
def test_pool_keys_grid_bruteforce_and_special_cases(oracle):
    cfg = SMALL
    L = _layer(cfg)
    R, Nb, _, S, D = L["kv"].shape
    grid = oracle.pool_keys_grid(L["kv"])
    T = Nb * S
    assert grid.shape == (R, T // 16, D)
    keys = bf.bits_to_f64(L["kv"][:, :, 0]).reshape(R, T, D)
    n_comp = (T - 32) // 16 + 1
    for j in (0, 1, 5, n_comp - 1):
        want = bf.f64_to_bf16_bits(keys[:, 16 * j:16 * j + 32].mean(axis=1))        # numpy mean, independent of the loops
        assert np.max(np.abs(grid[:, j].astype(np.int32) - want.astype(np.int32))) <= 1
    assert np.all(grid[:, n_comp:] == 0)                                           # windows crossing the end do not exist
    # window = stride = S reduces to o1 (one key per block)
    np.testing.assert_array_equal(oracle.pool_keys_grid(L["kv"], window=S, stride=S), oracle.pool_keys(L["kv"]))
    # a constant context pools to that constant
    const = L["kv"].copy()
    const[:, :, 0] = const[:, :1, 0, :1]
    g2 = oracle.pool_keys_grid(const)
    assert np.all(g2[:, :n_comp] == const[:, :1, 0, 0])


def test_select_grid_bruteforce_forced_blocks_and_needle(oracle):
    rng = np.random.default_rng(11)
    cfg = SMALL.with_(n_blocks=20)
    L = _layer(cfg)
    grid = oracle.pool_keys_grid(L["kv"])
    R, Nb = cfg.rows, cfg.n_blocks
    s = bf.bits_to_f64(L["F"])[:, None, :] * bf.bits_to_f64(grid)
    s = s.sum(-1)                                                                   # [R][4 Nb] fp64, brute force
    for n_cand, n_init, n_local, k in [(20, 1, 4, 9), (20, 0, 0, 5), (13, 2, 3, 7), (6, 1, 4, 9), (3, 1, 4, 9)]:
        ids, bs = oracle.forecast_select_grid(L["F"], grid, k, n_cand, n_init, n_local)
        for r in range(R):
            block = [max(s[r, j] for j in range(4 * b, 4 * b + 4) if j < 4 * n_cand - 1) for b in range(n_cand)]
            forced = set(b for b in range(n_cand) if b < n_init or b >= n_cand - n_local)
            got = [int(x) for x in ids[r] if x >= 0]
            assert got == sorted(got) and forced <= set(got) and len(got) == min(k, n_cand)
            rest = sorted((b for b in range(n_cand) if b not in forced), key=lambda b: (-block[b], b))
            assert set(got) - forced == set(rest[:max(0, min(k, n_cand) - len(forced))])
    # needle: keys equal to 8 F only in tokens [64 b + 16, 64 b + 48) -- exactly window 4b+1 -- pull block b in, and the
    # window that starts in block b-1 and reaches into b (j = 4b - 1) does not pull block b-1 above it
    b = 9
    kv = L["kv"].copy()
    needle = bf.f64_to_bf16_bits(8.0 * bf.bits_to_f64(L["F"]))
    kv[:, b, 0, 16:48] = needle[:, None, :]
    ids, bs = oracle.forecast_select_grid(L["F"], oracle.pool_keys_grid(kv), 3, Nb, 0, 0)
    assert all(b in ids[r] for r in range(R)) and np.all(bs[:, b] > bs[:, b - 1])


# ---------------------------------------------------------------- closed forms the paper prints
def test_paper_closed_forms_golden():
    """tests/golden/paper_closed_forms.txt: P:L95 (33.5M Forecast parameters, 0.41% of 8B) and the
    KV-size figures of BASELINE.json configs 3-4; they fix 'one Forecast head of width D per KV head',
    the 8B GQA shape and the block-major KV layout sizes used by synth."""
    vals = {}
    with open(os.path.join(GOLDEN, "paper_closed_forms.txt")) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                key, v = line.split("=")
                vals[key.strip()] = float(v)
    c = synth.CFG3_128K
    hidden = 4096
    n_proj = c.n_layers                 # 31 lookahead projections + the layer-0 same-layer one
    params = hidden * c.n_kv_heads * c.head_dim * n_proj
    assert abs(params / 1e6 - vals["forecast_params_millions"]) < 0.1          # P:L95 prints 33.5M
    assert 7.9e9 < params / (vals["forecast_params_percent_of_8b"] / 100) < 8.4e9      # "of the 8B total"
    per_seq = c.n_layers * c.kv_bytes_per_layer / c.batch
    assert round(per_seq / 1e9, 1) == vals["kv_gb_per_sequence_128k"]
    assert round(synth.CFG4_128K.n_layers * synth.CFG4_128K.kv_bytes_per_layer / 1e9) == vals["kv_gb_batch32_128k"]
    assert c.block_bytes == 32 * 1024 and c.context == 131072 and synth.CFG2_32K.context == 32768
    assert synth.CFG1_TINY.context == 4096 and synth.CFG1_TINY.block_bytes == 16 * 1024


# ---------------------------------------------------------------- o16: attention over a partly filled newest block
def test_sparse_attn_len_all_blocks_plus_tail_is_dense_attention_over_T_tokens(oracle):
    """(o16 pin 1) Every complete block + the open block listed, seq_len = 64 n + r per row  =>  dense softmax attention over
    the first seq_len[r] tokens of the row: torch's scaled_dot_product_attention on the flattened token axis (a library
    routine that knows nothing about blocks) and an independent numpy softmax.  Rows have different lengths; one ends exactly
    on a block boundary, one holds a single token.  Pins Alg.2 l.2 (the appended token is attended) + Eq.5."""
    L = _layer(SMALL)
    R, Nb, _, S, D = L["kv"].shape
    B, Hq, G, Hkv = SMALL.batch, SMALL.n_q_heads, SMALL.group, SMALL.n_kv_heads
    seq_len = np.array([5 * S + 17, 7 * S, 1, Nb * S - 1], dtype=np.int64)[:R]
    assert len(seq_len) == R
    ids = np.tile(np.arange(Nb, dtype=np.int32), (R, 1))              # every block: those beyond seq_len must contribute nothing
    O, O64 = oracle.sparse_attn_len(L["Q"], L["kv"], ids, seq_len, pool_is_indexed=True)
    kvf = bf.bits_to_f64(L["kv"])
    Qf = bf.bits_to_f64(L["Q"])
    for r in range(R):
        b, g = divmod(r, Hkv)
        T = int(seq_len[r])
        K = kvf[r, :, 0].reshape(Nb * S, D)[:T]
        V = kvf[r, :, 1].reshape(Nb * S, D)[:T]
        q = Qf[b, g * G:(g + 1) * G]
        z = q @ K.T / np.sqrt(D)
        p = np.exp(z - z.max(axis=1, keepdims=True))
        p /= p.sum(axis=1, keepdims=True)
        np.testing.assert_allclose(O64[b, g * G:(g + 1) * G], p @ V, rtol=0, atol=1e-12)
        ref = torch.nn.functional.scaled_dot_product_attention(torch.from_numpy(q).reshape(1, G, 1, D), torch.from_numpy(K).expand(1, G, T, D),
                                                               torch.from_numpy(V).expand(1, G, T, D))
        np.testing.assert_allclose(O64[b, g * G:(g + 1) * G], ref.reshape(G, D).numpy(), rtol=0, atol=1e-12)
    np.testing.assert_array_equal(O, bf.f64_to_bf16_bits(np.where(np.abs(O64) < 1e-30, 0.0, O64)))


def test_sparse_attn_len_reduces_to_o6_and_ignores_what_lies_behind_the_tail(oracle):
    """(o16 pins 2-5) seq_len = Nb * S (every block complete) reproduces o6 bit for bit in both pool forms; tokens behind
    seq_len are never read (NaN there changes nothing); a listed block that lies wholly beyond seq_len counts like id -1; a row
    with seq_len 0 gives O = 0; a tail of one token with V = c for that token alone gives O = c."""
    L = _layer(SMALL)
    R, Nb, _, S, D = L["kv"].shape
    kp = oracle.pool_keys(L["kv"])
    ids, _ = oracle.forecast_select(L["F"], kp, SMALL.topk)
    ids[1, -2:] = -1
    pool = oracle.gather(L["kv"], ids)
    full = np.full(R, Nb * S, dtype=np.int64)
    O6, O6_64 = oracle.sparse_attn(L["Q"], pool, ids)
    Ol, Ol64 = oracle.sparse_attn_len(L["Q"], pool, ids, full)
    np.testing.assert_array_equal(Ol, O6)
    np.testing.assert_allclose(Ol64, O6_64, rtol=0, atol=1e-12)
    Oi, _ = oracle.sparse_attn_len(L["Q"], L["kv"], ids, full, pool_is_indexed=True)
    np.testing.assert_array_equal(Oi, O6)
    # the open block is the highest listed id of each row; cut it to 9 tokens and poison what lies behind
    seq_len = np.array([int(ids[r][ids[r] >= 0].max()) * S + 9 for r in range(R)], dtype=np.int64)
    kv_nan = L["kv"].copy()
    for r in range(R):
        j = int(seq_len[r]) // S
        kv_nan[r, j, :, 9:] = 0x7FC0                                  # NaN behind the tail, K and V
        kv_nan[r, j + 1:] = 0x7FC0                                    # and in every later block
    Oa, Oa64 = oracle.sparse_attn_len(L["Q"], L["kv"], ids, seq_len, pool_is_indexed=True)
    Ob, Ob64 = oracle.sparse_attn_len(L["Q"], kv_nan, ids, seq_len, pool_is_indexed=True)
    assert np.all(np.isfinite(Ob64))
    np.testing.assert_array_equal(Oa, Ob)
    assert not np.array_equal(Oa, O6), "cutting the newest block to 9 tokens must change O"
    want = np.zeros_like(Oa64)
    Qf, kvf = bf.bits_to_f64(L["Q"]), bf.bits_to_f64(L["kv"])
    for b in range(SMALL.batch):
        for h in range(SMALL.n_q_heads):
            r = b * SMALL.n_kv_heads + h // SMALL.group
            toks = [(j, t) for j in ids[r] if j >= 0 for t in range(S) if j * S + t < seq_len[r]]
            K = np.stack([kvf[r, j, 0, t] for j, t in toks])
            V = np.stack([kvf[r, j, 1, t] for j, t in toks])
            z = K @ Qf[b, h] / np.sqrt(D)
            p = np.exp(z - z.max())
            want[b, h] = (p / p.sum()) @ V
    np.testing.assert_allclose(Oa64, want, rtol=0, atol=1e-12)
    # a listed block wholly beyond seq_len == that slot set to -1
    ids_cut = ids.copy()
    short = seq_len - 9 - S                                           # the open block and the one before it lie beyond
    for r in range(R):
        ids_cut[r][ids[r] * S >= short[r]] = -1
    Oc, _ = oracle.sparse_attn_len(L["Q"], L["kv"], ids, short, pool_is_indexed=True)
    Od, _ = oracle.sparse_attn(L["Q"], L["kv"], ids_cut, pool_is_indexed=True)
    np.testing.assert_array_equal(Oc, Od)
    # empty rows -> zeros; a single attended token -> its V row exactly
    Oz, Oz64 = oracle.sparse_attn_len(L["Q"], L["kv"], ids, np.zeros(R, dtype=np.int64), pool_is_indexed=True)
    assert not Oz.any() and not Oz64.any()
    one = np.tile(np.array([[0] + [-1] * (SMALL.topk - 1)], dtype=np.int32), (R, 1))
    O1, _ = oracle.sparse_attn_len(L["Q"], L["kv"], one, np.ones(R, dtype=np.int64), pool_is_indexed=True)
    for b in range(SMALL.batch):
        for h in range(SMALL.n_q_heads):
            np.testing.assert_array_equal(O1[b, h], L["kv"][b * SMALL.n_kv_heads + h // SMALL.group, 0, 1, 0])
