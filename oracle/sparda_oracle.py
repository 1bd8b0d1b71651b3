"""numpy/ctypes wrapper around ``sparda_oracle.c`` -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

o1-o9: argument marshalling only; every number is computed by the plain C loops in ``sparda_oracle.c`` (which cites
the paper passage each function follows).  Written here, as plain Python / numpy loops that call those:
``decode_pipeline`` (o10: Algorithm 2 lines 4-7, strictly in order), ``reuse_plan`` /
``decode_pipeline_cached`` (o11 / o12: the previous-step block cache, reading q18), ``append_kv`` (o13: Algorithm 2
lines 2-3) and ``pool_keys_grid`` / ``forecast_select_grid`` (o14 / o15: the (32,16) compressed-key grid with
the max-pool to blocks, reading q19 -- PARITY UNPINNED BY THE PAPER, which does not state the pooling geometry) and
``sparse_attn_len`` (o16: Eq.5 over a cache whose last block is partly filled, Algorithm 2 line 2 P:L300 + Eq.1 P:L53-56,
reading q7).
Every function is pinned in ``tests/test_oracle_pins.py``.

bf16 tensors are numpy ``uint16`` arrays holding the raw upper halves of fp32 values.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sparda_oracle.c")
_LIB = os.path.join(_HERE, "libsparda_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C11 + OpenMP over independent units)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-std=c11", "-O2", "-fopenmp", "-fPIC", "-shared", "-fno-fast-math",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.sparda_oracle_bf16_to_double.restype = ctypes.c_double
        _lib.sparda_oracle_bf16_to_double.argtypes = [ctypes.c_uint16]
        _lib.sparda_oracle_double_to_bf16.restype = ctypes.c_uint16
        _lib.sparda_oracle_double_to_bf16.argtypes = [ctypes.c_double]
        _lib.sparda_oracle_threads.restype = ctypes.c_int
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


def _u16(a) -> np.ndarray:
    a = np.ascontiguousarray(a)
    assert a.dtype == np.uint16, a.dtype
    return a


def _i64(x):
    return ctypes.c_int64(int(x))


def _i32(x):
    return ctypes.c_int(int(x))


def threads() -> int:
    return int(_load().sparda_oracle_threads())


def set_threads(n: int) -> None:
    _load().sparda_oracle_set_threads(_i32(n))


# ---- bf16 helpers -------------------------------------------------------------------------
def bf16_bits_to_f64(a: np.ndarray) -> np.ndarray:
    """Exact widening of raw bf16 bits to float64 (numpy only, used by tests and callers)."""
    a = np.ascontiguousarray(a, dtype=np.uint16)
    return (a.astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def double_to_bf16(x: float) -> int:
    return int(_load().sparda_oracle_double_to_bf16(ctypes.c_double(x)))


def from_torch(t) -> np.ndarray:
    """torch.bfloat16 CPU tensor -> uint16 bits (no copy of values, no arithmetic)."""
    import torch
    assert t.dtype == torch.bfloat16 and t.device.type == "cpu"
    return t.contiguous().view(torch.int16).numpy().view(np.uint16)


def to_torch(a: np.ndarray):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int16)).view(torch.bfloat16)


# ---- o1 .. o9 -----------------------------------------------------------------------------
def pool_keys(kv: np.ndarray) -> np.ndarray:
    """o1 (Eq.2, kernel = stride = S).  kv [R][Nb][2][S][D] -> Kpool [R][Nb][D]."""
    kv = _u16(kv)
    R, Nb, two, S, D = kv.shape
    assert two == 2
    out = np.empty((R, Nb, D), dtype=np.uint16)
    _load().sparda_oracle_pool_keys(_p(kv), _i64(R), _i64(Nb), _i32(S), _i32(D), _p(out))
    return out


def forecast_project(X: np.ndarray, WF: np.ndarray, Hkv: int, D: int) -> np.ndarray:
    """o2 (Eq.3).  X [B][hidden], WF [hidden][Hkv*D] -> F [B*Hkv][D]."""
    X, WF = _u16(X), _u16(WF)
    B, hidden = X.shape
    assert WF.shape == (hidden, Hkv * D)
    out = np.empty((B * Hkv, D), dtype=np.uint16)
    _load().sparda_oracle_forecast_project(_p(X), _p(WF), _i64(B), _i64(hidden), _i32(Hkv), _i32(D), _p(out))
    return out


def score(F: np.ndarray, kpool: np.ndarray) -> np.ndarray:
    """o3 (Eq.4).  F [R][D], Kpool [R][Nb][D] -> s [R][Nb] fp32."""
    F, kpool = _u16(F), _u16(kpool)
    R, Nb, D = kpool.shape
    assert F.shape == (R, D)
    out = np.empty((R, Nb), dtype=np.float32)
    _load().sparda_oracle_score(_p(F), _p(kpool), _i64(R), _i64(Nb), _i32(D), _p(out))
    return out


def topk(scores: np.ndarray, k: int, n_cand: int | None = None) -> np.ndarray:
    """o4 (P:L78 f_top).  s [R][Nb] fp32 -> ids [R][k] int32 ascending, -1 padded."""
    scores = np.ascontiguousarray(scores, dtype=np.float32)
    R, Nb = scores.shape
    n_cand = Nb if n_cand is None else n_cand
    assert 0 <= n_cand <= Nb
    out = np.empty((R, k), dtype=np.int32)
    _load().sparda_oracle_topk(_p(scores), _i64(R), _i64(Nb), _i64(n_cand), _i32(k), _p(out))
    return out


def forecast_select(F: np.ndarray, kpool: np.ndarray, k: int, n_cand: int | None = None):
    """o3 + o4: returns (ids, scores)."""
    s = score(F, kpool)
    return topk(s, k, n_cand), s


def gather(kv: np.ndarray, ids: np.ndarray, pool: np.ndarray | None = None) -> np.ndarray:
    """o5.  kv [R][Nb][2][S][D], ids [R][k] -> pool [R][k][2][S][D]; -1 slots untouched."""
    kv = _u16(kv)
    ids = np.ascontiguousarray(ids, dtype=np.int32)
    R, Nb, two, S, D = kv.shape
    k = ids.shape[1]
    assert ids.shape[0] == R
    if pool is None:
        pool = np.zeros((R, k, 2, S, D), dtype=np.uint16)
    assert pool.shape == (R, k, 2, S, D) and pool.dtype == np.uint16 and pool.flags.c_contiguous
    _load().sparda_oracle_gather(_p(kv), _p(ids), _i64(R), _i64(Nb), _i32(k), _i32(S), _i32(D), _p(pool))
    return pool


def sparse_attn(Q: np.ndarray, pool: np.ndarray, ids: np.ndarray, pool_is_indexed: bool = False):
    """o6 (Eq.5).  Q [B][Hq][D], pool [R][n_slots][2][S][D], ids [R][k] -> (O bf16 bits, O float64)."""
    Q, pool = _u16(Q), _u16(pool)
    ids = np.ascontiguousarray(ids, dtype=np.int32)
    B, Hq, D = Q.shape
    R, n_slots, two, S, D2 = pool.shape
    assert two == 2 and D2 == D and R % B == 0
    Hkv = R // B
    k = ids.shape[1]
    assert ids.shape[0] == R
    if not pool_is_indexed:
        assert n_slots == k
    else:
        assert ids.max(initial=-1) < n_slots
    O = np.empty((B, Hq, D), dtype=np.uint16)
    O64 = np.empty((B, Hq, D), dtype=np.float64)
    _load().sparda_oracle_sparse_attn(_p(Q), _p(pool), _p(ids), _i32(1 if pool_is_indexed else 0), _i64(B), _i32(Hq),
                                      _i32(Hkv), _i32(D), _i32(S), _i32(k), _i64(n_slots), _p(O), _p(O64))
    return O, O64


def dense_attn(Q: np.ndarray, kv: np.ndarray):
    """o7 (textbook).  Q [B][Hq][D], kv [R][Nb][2][S][D] -> (O bf16 bits, O float64)."""
    Q, kv = _u16(Q), _u16(kv)
    B, Hq, D = Q.shape
    R, Nb, two, S, D2 = kv.shape
    assert two == 2 and D2 == D and R % B == 0
    O = np.empty((B, Hq, D), dtype=np.uint16)
    O64 = np.empty((B, Hq, D), dtype=np.float64)
    _load().sparda_oracle_dense_attn(_p(Q), _p(kv), _i64(B), _i32(Hq), _i32(R // B), _i32(D), _i32(S), _i64(Nb),
                                     _p(O), _p(O64))
    return O, O64


def prefill_select(F: np.ndarray, kpool: np.ndarray, k: int, row0: int = 0, n_rows: int | None = None,
                   S: int = 64, want_scores: bool = False):
    """o8 (Alg.1 l.2, causal rule q8).  F [Hkv][T][D], Kpool [Hkv][Nb][D] -> ids [Hkv][n_rows][k]."""
    F, kpool = _u16(F), _u16(kpool)
    Hkv, T, D = F.shape
    Nb = kpool.shape[1]
    assert kpool.shape == (Hkv, Nb, D)
    n_rows = T - row0 if n_rows is None else n_rows
    assert 0 <= row0 and row0 + n_rows <= T
    ids = np.empty((Hkv, n_rows, k), dtype=np.int32)
    sc = np.empty((Hkv, n_rows, Nb), dtype=np.float32) if want_scores else None
    _load().sparda_oracle_prefill_select(_p(F), _p(kpool), _i32(Hkv), _i64(T), _i64(Nb), _i32(D), _i32(S),
                                         _i64(row0), _i64(n_rows), _i32(k), _p(ids),
                                         _p(sc) if want_scores else None)
    return (ids, sc) if want_scores else ids


def prefill_select_baseline(Q: np.ndarray, kpool: np.ndarray, k: int, row0: int = 0, n_rows: int | None = None,
                            S: int = 64, want_scores: bool = False):
    """o9 (Eq.6 left).  Q [Hq][T][D], Kpool [Hkv][Nb][D] -> ids [Hkv][n_rows][k]."""
    Q, kpool = _u16(Q), _u16(kpool)
    Hq, T, D = Q.shape
    Hkv, Nb, _ = kpool.shape
    assert Hq % Hkv == 0
    n_rows = T - row0 if n_rows is None else n_rows
    ids = np.empty((Hkv, n_rows, k), dtype=np.int32)
    sc = np.empty((Hkv, n_rows, Nb), dtype=np.float32) if want_scores else None
    _load().sparda_oracle_prefill_select_baseline(_p(Q), _p(kpool), _i32(Hq), _i32(Hkv), _i64(T), _i64(Nb), _i32(D),
                                                  _i32(S), _i64(row0), _i64(n_rows), _i32(k), _p(ids),
                                                  _p(sc) if want_scores else None)
    return (ids, sc) if want_scores else ids


# ---- o10 ----------------------------------------------------------------------------------
def decode_pipeline(layers, k: int):
    """o10: Algorithm 2 lines 4-7 for L layers, strictly in order, no overlap.

    ``layers`` is a list of dicts with uint16 arrays ``kv`` [R][Nb][2][S][D], ``kpool`` [R][Nb][D],
    ``F`` [R][D], ``Q`` [B][Hq][D]; layer 0 additionally has ``F0cur`` [R][D].
    Layer 0: same-layer selection with F0cur, attention straight from its own cache.
    Layer l >= 1: ids_l = f_top(F_{l-1} Kpool_l^T, k) (reading q9); gather; attention.
    F of the last layer is unused.  Returns per-layer dicts {ids, scores, pool, O, O64}.
    """
    out = []
    for l, lay in enumerate(layers):
        f = lay["F0cur"] if l == 0 else layers[l - 1]["F"]
        ids, s = forecast_select(f, lay["kpool"], k)
        if l == 0:
            pool = None
            O, O64 = sparse_attn(lay["Q"], lay["kv"], ids, pool_is_indexed=True)
        else:
            pool = gather(lay["kv"], ids)
            O, O64 = sparse_attn(lay["Q"], pool, ids, pool_is_indexed=False)
        out.append({"ids": ids, "scores": s, "pool": pool, "O": O, "O64": O64})
    return out


# ---- o11 / o12: step-to-step block reuse ----------------------------------
def reuse_plan(ids_new: np.ndarray, slot_ids: np.ndarray):
    """o11: which pool slot holds which block after a step, and what must be fetched.

    The paper's engine keeps, per layer, the blocks selected at the previous decode step and fetches
    "only newly selected blocks"; it gives no slot policy.  Reading q18: a slot
    whose block is selected again keeps it; the j-th smallest newly selected block id that is not
    resident goes to the j-th lowest-numbered slot whose block was not selected again; slots left
    over (fewer selected blocks than slots) become empty (-1).  Plain loops over Python sets, one
    row at a time.

    ids_new [R][k] (ascending, -1 padded), slot_ids [R][k] (block held by each slot, -1 = empty)
    -> (slot_ids_after [R][k], fetch [R][k]): fetch[r][s] = block to copy into slot s, or -1.
    """
    ids_new = np.asarray(ids_new, dtype=np.int32)
    slot_ids = np.asarray(slot_ids, dtype=np.int32)
    assert ids_new.shape == slot_ids.shape
    R, k = ids_new.shape
    after = np.full((R, k), -1, dtype=np.int32)
    fetch = np.full((R, k), -1, dtype=np.int32)
    for r in range(R):
        wanted = [int(b) for b in ids_new[r] if b >= 0]
        wanted_set = set(wanted)
        resident = set()
        free = []
        for s in range(k):
            b = int(slot_ids[r, s])
            if b >= 0 and b in wanted_set and b not in resident:
                after[r, s] = b
                resident.add(b)
            else:
                free.append(s)
        misses = sorted(b for b in wanted_set if b not in resident)
        assert len(misses) <= len(free)
        for j, b in enumerate(misses):
            after[r, free[j]] = b
            fetch[r, free[j]] = b
    return after, fetch


def decode_pipeline_cached(steps, k: int, state=None):
    """o12: Algorithm 2 lines 4-7 over several decode steps with the per-layer block cache of the
    previous step.  ``steps`` is a list (one entry per decode step) of layer lists as in
    ``decode_pipeline``; the KV caches and pooled keys may be shared between steps.  Per layer l >= 1 the pool
    persists between steps: o11 decides the slots, o5 copies only the fetched blocks, o6 attends over the pool
    in slot order.  Returns (per-step list of per-layer dicts {ids, slot_ids, fetch, pool, O, O64}, state)."""
    n_layers = len(steps[0])
    if state is None:
        state = {"slot_ids": [None] * n_layers, "pool": [None] * n_layers}
    out = []
    for layers in steps:
        res = []
        for l, lay in enumerate(layers):
            f = lay["F0cur"] if l == 0 else layers[l - 1]["F"]
            ids, s = forecast_select(f, lay["kpool"], k)
            if l == 0:
                O, O64 = sparse_attn(lay["Q"], lay["kv"], ids, pool_is_indexed=True)
                res.append({"ids": ids, "scores": s, "slot_ids": None, "fetch": None, "pool": None, "O": O, "O64": O64})
                continue
            if state["slot_ids"][l] is None:
                R, _, _, S, D = lay["kv"].shape
                state["slot_ids"][l] = np.full((R, k), -1, dtype=np.int32)
                state["pool"][l] = np.zeros((R, k, 2, S, D), dtype=np.uint16)
            after, fetch = reuse_plan(ids, state["slot_ids"][l])
            gather(lay["kv"], fetch, state["pool"][l])       # copies fetch >= 0 slots only
            state["slot_ids"][l] = after
            O, O64 = sparse_attn(lay["Q"], state["pool"][l], after, pool_is_indexed=False)
            res.append({"ids": ids, "scores": s, "slot_ids": after.copy(), "fetch": fetch, "pool": state["pool"][l].copy(),
                        "O": O, "O64": O64})
        out.append(res)
    return out, state


# ---- o13: decode-time cache maintenance -----------------------------------
def append_kv(kv: np.ndarray, kpool: np.ndarray, k_new: np.ndarray, v_new: np.ndarray, t: int):
    """o13: Algorithm 2 lines 2-3: append the new token's K and V at position t of every row's cache and
    "update K~ incrementally": when the token completes block j = t // S (t % S == S - 1) the block's pooled
    key becomes the mean of its S keys (Eq.2, kernel = stride = S; computed by o1 on the finished block).

    kv [R][Nb][2][S][D] and kpool [R][Nb][D] are modified in place; k_new, v_new [R][D] (bf16 bits).
    Returns the number of complete blocks after the append, (t + 1) // S: the candidate range of the next selection."""
    kv, kpool = _u16(kv), _u16(kpool)
    R, Nb, two, S, D = kv.shape
    j, o = divmod(int(t), S)
    assert 0 <= j < Nb and k_new.shape == (R, D) and v_new.shape == (R, D)
    for r in range(R):
        kv[r, j, 0, o, :] = k_new[r]
        kv[r, j, 1, o, :] = v_new[r]
    if o == S - 1:
        done = pool_keys(np.ascontiguousarray(kv[:, j:j + 1]))       # o1 on the finished block only
        kpool[:, j, :] = done[:, 0, :]
    return (int(t) + 1) // S


# ---- o14 / o15: the paper's selector geometry -- PARITY UNPINNED BY THE PAPER ------
# The paper compresses keys with overlapping windows (l_C, s) = (32, 16) (Eq.2) and says f_top
# "max-pools compressed-key-grid scores to block-level scores" without giving the pooling kernel, stride or
# padding.  Reading q19: compressed key j covers tokens [16 j, 16 j + 32), j = 0 .. T/16 - 2;
# block b's score is the maximum over the compressed keys whose window STARTS inside the block (j = 4b .. 4b+3, the
# last one reaching 16 tokens into the next block; block Nb-1 has three).  Initial and local blocks do not take part
# in the ranking and are always attended (Eq.1): B = init U local U top-k.  These two functions are
# pinned to brute force and invariants written independently in tests/, not to anything the paper prints.
def pool_keys_grid(kv: np.ndarray, window: int = 32, stride: int = 16) -> np.ndarray:
    """o14 (Eq.2, P:L60 with (l_C, s) = (32, 16)): Kgrid[r, j, :] = bf16(mean of keys stride*j .. stride*j+window-1),
    fp64 sum in ascending token order.  kv [R][Nb][2][S][D] -> Kgrid [R][Nb*S/stride][D]; rows j >= n_comp =
    (T - window)/stride + 1 (windows that would cross the end of the context) are zero."""
    kv = _u16(kv)
    R, Nb, two, S, D = kv.shape
    T = Nb * S
    n_rows, n_comp = T // stride, (T - window) // stride + 1
    keys = bf16_bits_to_f64(kv[:, :, 0]).reshape(R, T, D)
    out = np.zeros((R, n_rows, D), dtype=np.uint16)
    for r in range(R):
        for j in range(n_comp):
            acc = np.zeros(D, dtype=np.float64)
            for t in range(stride * j, stride * j + window):
                acc += keys[r, t]
            mean = acc / window
            out[r, j] = [double_to_bf16(float(x)) for x in mean]
    return out


def forecast_select_grid(F: np.ndarray, kgrid: np.ndarray, k_total: int, n_cand: int, n_init: int, n_local: int, per_block: int = 4):
    """o15 (Eq.1, Eq.4, f_top P:L78, reading q19): compressed-key scores s_j = F . Kgrid_j (o3), block score =
    max of the per_block compressed keys that start in the block and exist (j < per_block * n_cand - 1), blocks
    [0, n_init) and [n_cand - n_local, n_cand) always selected, the other k_total - n_init - n_local picked by block score
    (o4: score descending, lowest id on ties) among the remaining candidates; ascending ids, -1 padded.
    Returns (ids [R][k_total], block_scores [R][n_cand] fp32 with forced blocks at +inf)."""
    s = score(F, kgrid)                                       # [R][n_rows] fp32, raw logits
    R = s.shape[0]
    n_keys = per_block * n_cand - 1
    ids = np.full((R, k_total), -1, dtype=np.int32)
    bs = np.full((R, max(n_cand, 0)), -np.inf, dtype=np.float32)
    for r in range(R):
        for b in range(n_cand):
            js = [j for j in range(per_block * b, per_block * b + per_block) if j < n_keys]
            bs[r, b] = max(s[r, j] for j in js)
        forced = [b for b in range(n_cand) if b < n_init or b >= n_cand - n_local]
        assert len(forced) <= k_total
        free = [b for b in range(n_cand) if b not in forced]
        free.sort(key=lambda b: (-float(bs[r, b]), b))
        chosen = sorted(forced + free[:k_total - len(forced)])
        ids[r, :len(chosen)] = chosen
        for b in forced:
            bs[r, b] = np.inf
    return ids, bs


def sparse_attn_len(Q: np.ndarray, pool: np.ndarray, ids: np.ndarray, seq_len: np.ndarray, pool_is_indexed: bool = False):
    """o16: o6 (Eq.5) over the tokens that exist.  Row r's cache holds seq_len[r] tokens: the new token's K / V is appended
    before the attention (Alg.2 l.2) and the local window that holds it is always attended (Eq.1), so the
    newest block is in general partly filled (reading q7).  Block j of row r holds the tokens S*j .. S*j + S - 1; it contributes
    its first min(S, seq_len[r] - S*j) tokens, nothing when that is <= 0; whatever bytes sit behind them in the block are
    never read.  Otherwise Eq.5 as in o6: z_t = q . k_t / sqrt(D), softmax over every contributing token of every
    listed block (id >= 0), O = sum_t p_t v_t; fp64 throughout, one rounding to bf16.  A head with no token gives O = 0.
    Q [B][Hq][D], pool [R][n_slots][2][S][D] (slot i holds block ids[r][i], or the cache addressed by id when
    pool_is_indexed), ids [R][k] (block ids, -1 = none), seq_len [R] -> (O bf16 bits, O float64).  Plain loops; small cases."""
    Q, pool = _u16(Q), _u16(pool)
    ids = np.ascontiguousarray(ids, dtype=np.int32)
    seq_len = np.ascontiguousarray(seq_len, dtype=np.int64)
    B, Hq, D = Q.shape
    R, n_slots, two, S, D2 = pool.shape
    assert two == 2 and D2 == D and R % B == 0 and ids.shape[0] == R and seq_len.shape == (R,)
    Hkv = R // B
    G = Hq // Hkv
    k = ids.shape[1]
    assert n_slots == k or pool_is_indexed
    Qf = bf16_bits_to_f64(Q)
    O64 = np.zeros((B, Hq, D), dtype=np.float64)
    O = np.zeros((B, Hq, D), dtype=np.uint16)
    for b in range(B):
        for h in range(Hq):
            r = b * Hkv + h // G
            z, vs = [], []
            for i in range(k):
                j = int(ids[r, i])
                if j < 0:
                    continue
                n_tok = min(S, int(seq_len[r]) - S * j)
                if n_tok <= 0:
                    continue
                blk = pool[r, j if pool_is_indexed else i]
                Kt = bf16_bits_to_f64(blk[0, :n_tok])
                Vt = bf16_bits_to_f64(blk[1, :n_tok])
                for t in range(n_tok):
                    z.append(float(np.dot(Qf[b, h], Kt[t])) / np.sqrt(float(D)))
                    vs.append(Vt[t])
            if not z:
                continue
            z = np.array(z)
            pr = np.exp(z - z.max())
            pr = pr / pr.sum()
            acc = np.zeros(D)
            for t in range(len(z)):
                acc += pr[t] * vs[t]
            O64[b, h] = acc
            O[b, h] = [double_to_bf16(float(x)) for x in acc]
    return O, O64
