"""Thin ctypes binding of libsparda (include/sparda.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI.  torch is used for device / pinned
memory and streams.  There is no fallback: if ``libsparda.so`` is missing or a call fails, a
``SpardaError`` is raised.
"""
from __future__ import annotations

import ctypes
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsparda.so")

GATHER_TMA, GATHER_LDG = 0, 1
STEP_OVERLAP, STEP_SERIAL = 0, 1

EXPORTS = [
    "sparda_create", "sparda_destroy", "sparda_pool_keys", "sparda_forecast_project", "sparda_append_kv", "sparda_pool_keys_grid", "sparda_forecast_select_grid", "sparda_forecast_select", "sparda_prefetch_launch",
    "sparda_sparse_decode", "sparda_sparse_decode_varlen", "sparda_sparse_decode_noalloc", "sparda_noalloc_last_error", "sparda_decode_step", "sparda_decode_step_host", "sparda_profile_enable",
    "sparda_reuse_plan", "sparda_forecast_select_plan", "sparda_decode_step_cached",
    "sparda_profile_read", "sparda_prefill_select", "sparda_prefill_select_baseline",
    "sparda_probe_launch", "sparda_set_layer_standin", "sparda_enable_peer_tier", "sparda_set_step_candidates", "sparda_set_step_selector",
    "sparda_launch_count", "sparda_tmap_encodes", "sparda_get_select_cluster", "sparda_get_attn_cluster", "sparda_get_attn_splits", "sparda_get_gather_ctas", "sparda_strerror",
    "sparda_last_cuda_error", "sparda_version",
]


class SpardaError(RuntimeError):
    pass


class SpardaConfig(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int) for n in (
        "batch", "n_q_heads", "n_kv_heads", "head_dim", "block_size", "max_blocks", "topk", "gather_ctas",
        "gather_mode", "attn_splits", "max_layers", "select_cluster", "hidden", "attn_impl", "no_pdl")]


class SpardaLayer(ctypes.Structure):
    _fields_ = [("F", ctypes.c_void_p), ("Q", ctypes.c_void_p), ("Kpool", ctypes.c_void_p), ("kv", ctypes.c_void_p),
                ("O", ctypes.c_void_p), ("ids", ctypes.c_void_p), ("X", ctypes.c_void_p), ("WF", ctypes.c_void_p),
                ("WFcur", ctypes.c_void_p)]


class SpardaCachedLayer(ctypes.Structure):
    _fields_ = [("base", SpardaLayer), ("pool", ctypes.c_void_p), ("slot_ids", ctypes.c_void_p), ("fetch", ctypes.c_void_p),
                ("n_fetch", ctypes.c_void_p)]


_lib = None


def lib() -> ctypes.CDLL:
    """Load libsparda.so (built in-tree by ``build.build()``); fail loudly if it is not there."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise SpardaError(f"{LIB_PATH} not found: build it with `python -m paper_2606_04511_b200.build` "
                              "(there is no CPU or PyTorch fallback)")
        L = ctypes.CDLL(LIB_PATH)
        vp, i32, i64 = ctypes.c_void_p, ctypes.c_int, ctypes.c_int64
        L.sparda_create.argtypes = [ctypes.POINTER(SpardaConfig), ctypes.POINTER(vp)]
        L.sparda_destroy.argtypes = [vp]
        L.sparda_pool_keys.argtypes = [vp, vp, i64, i32, vp, vp]
        L.sparda_pool_keys_grid.argtypes = [vp, vp, i64, i32, vp, vp]
        L.sparda_forecast_select_grid.argtypes = [vp, vp, vp, i32, i32, i32, i32, i32, vp, vp]
        L.sparda_forecast_project.argtypes = [vp, vp, vp, i32, vp, vp]
        L.sparda_append_kv.argtypes = [vp, vp, vp, i64, vp, i32, vp, vp, vp]
        L.sparda_forecast_select.argtypes = [vp, vp, vp, i32, i32, i32, vp, vp]
        L.sparda_prefetch_launch.argtypes = [vp, vp, i32, vp, i32, vp, vp]
        L.sparda_sparse_decode.argtypes = [vp, vp, vp, vp, i32, i32, i32, vp, vp]
        L.sparda_sparse_decode_varlen.argtypes = [vp, vp, vp, vp, vp, i32, i32, i32, vp, vp]
        L.sparda_sparse_decode_noalloc.argtypes = [i32, i32, i32, i32, vp, vp, vp, i32, i32, i32, vp, vp]
        L.sparda_noalloc_last_error.argtypes = []
        L.sparda_decode_step.argtypes = [vp, ctypes.POINTER(SpardaLayer), i32, vp, i32, i32, vp, vp, vp, vp, i32]
        L.sparda_decode_step_host.argtypes = L.sparda_decode_step.argtypes
        L.sparda_reuse_plan.argtypes = [vp, vp, i32, vp, vp, vp, vp]
        L.sparda_forecast_select_plan.argtypes = [vp, vp, vp, i32, i32, i32, vp, vp, vp, vp, vp]
        L.sparda_decode_step_cached.argtypes = [vp, ctypes.POINTER(SpardaCachedLayer), i32, vp, i32, i32, vp, vp, i32]
        L.sparda_profile_enable.argtypes = [vp, i32]
        L.sparda_profile_read.argtypes = [vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(i64)]
        L.sparda_prefill_select.argtypes = [vp, vp, vp, i32, i32, i32, i32, i32, vp, vp]
        L.sparda_prefill_select_baseline.argtypes = [vp, vp, vp, i32, i32, i32, i32, i32, vp, vp]
        L.sparda_launch_count.argtypes = [vp]
        L.sparda_launch_count.restype = i64
        L.sparda_probe_launch.argtypes = [vp, i32, vp, i64, vp]
        L.sparda_set_layer_standin.argtypes = [vp, vp, i64]
        L.sparda_enable_peer_tier.argtypes = [vp, i32]
        L.sparda_set_step_candidates.argtypes = [vp, i32]
        L.sparda_set_step_selector.argtypes = [vp, i32, i32, i32]
        L.sparda_tmap_encodes.argtypes = [vp]
        L.sparda_tmap_encodes.restype = i64
        L.sparda_get_select_cluster.argtypes = [vp]
        L.sparda_get_attn_cluster.argtypes = [vp]
        L.sparda_get_attn_splits.argtypes = [vp, i32]
        L.sparda_get_gather_ctas.argtypes = [vp]
        for f in ("sparda_strerror", "sparda_last_cuda_error", "sparda_version", "sparda_noalloc_last_error"):
            getattr(L, f).restype = ctypes.c_char_p
        L.sparda_strerror.argtypes = [i32]
        L.sparda_last_cuda_error.argtypes = [vp]
        _lib = L
    return _lib


def _ptr(t) -> int:
    if t is None:
        return 0
    if isinstance(t, int):
        return t
    assert t.is_contiguous(), "tensors crossing the C ABI must be contiguous"
    return t.data_ptr()


def _stream(s) -> int:
    if s is None:
        return torch.cuda.current_stream().cuda_stream
    return s.cuda_stream if hasattr(s, "cuda_stream") else int(s)


class Sparda:
    """One libsparda context (one shape family on the current device)."""

    def __init__(self, batch, n_q_heads, n_kv_heads, head_dim, max_blocks, topk, block_size=64, gather_ctas=0,
                 gather_mode=GATHER_TMA, attn_splits=0, max_layers=0, select_cluster=0, hidden=0, attn_impl=0, no_pdl=0):
        self._h = ctypes.c_void_p()
        self.cfg = SpardaConfig(batch, n_q_heads, n_kv_heads, head_dim, block_size, max_blocks, topk, gather_ctas,
                                gather_mode, attn_splits, max_layers, select_cluster, hidden, attn_impl, no_pdl)
        self._L = lib()
        rc = self._L.sparda_create(ctypes.byref(self.cfg), ctypes.byref(self._h))
        if rc != 0:
            self._h = ctypes.c_void_p()
            raise SpardaError(f"sparda_create: {self._L.sparda_strerror(rc).decode()}")
        self.rows = batch * n_kv_heads

    @classmethod
    def from_config(cls, cfg, **kw):
        return cls(cfg.batch, cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim, cfg.n_blocks, cfg.topk,
                   block_size=cfg.block_size, **kw)

    def close(self):
        if self._h:
            self._L.sparda_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc, what):
        if rc != 0:
            msg = self._L.sparda_strerror(rc).decode()
            if rc == -3:
                msg += ": " + self._L.sparda_last_cuda_error(self._h).decode()
            raise SpardaError(f"{what}: {msg}")

    # ---- entry points (same names as include/sparda.h without the prefix) ----
    def pool_keys(self, kv, n_rows, n_blocks, kpool, stream=None):
        self._check(self._L.sparda_pool_keys(self._h, _ptr(kv), n_rows, n_blocks, _ptr(kpool), _stream(stream)), "pool_keys")

    def pool_keys_grid(self, kv, n_rows, n_blocks, kgrid, stream=None):
        self._check(self._L.sparda_pool_keys_grid(self._h, _ptr(kv), n_rows, n_blocks, _ptr(kgrid), _stream(stream)), "pool_keys_grid")

    def forecast_select_grid(self, F, Kgrid, n_blocks, topk, ids_out, n_init=0, n_local=0, n_cand=None, stream=None):
        n_cand = n_blocks if n_cand is None else n_cand
        self._check(self._L.sparda_forecast_select_grid(self._h, _ptr(F), _ptr(Kgrid), n_blocks, n_cand, n_init, n_local, topk,
                                                        _ptr(ids_out), _stream(stream)), "forecast_select_grid")

    def forecast_project(self, X, WF, hidden, F_out, stream=None):
        self._check(self._L.sparda_forecast_project(self._h, _ptr(X), _ptr(WF), hidden, _ptr(F_out), _stream(stream)), "forecast_project")

    def append_kv(self, k_new, v_new, t, kv_cache, n_blocks, ksum, kpool, stream=None):
        self._check(self._L.sparda_append_kv(self._h, _ptr(k_new), _ptr(v_new), int(t), _ptr(kv_cache), n_blocks, _ptr(ksum),
                                             _ptr(kpool), _stream(stream)), "append_kv")

    def forecast_select(self, F, Kpool, n_blocks, topk, ids_out, n_cand=None, stream=None):
        n_cand = n_blocks if n_cand is None else n_cand
        self._check(self._L.sparda_forecast_select(self._h, _ptr(F), _ptr(Kpool), n_blocks, n_cand, topk, _ptr(ids_out),
                                                   _stream(stream)), "forecast_select")

    def prefetch_launch(self, host_kv, n_blocks, ids, topk, dev_pool, stream=None):
        self._check(self._L.sparda_prefetch_launch(self._h, _ptr(host_kv), n_blocks, _ptr(ids), topk, _ptr(dev_pool),
                                                   _stream(stream)), "prefetch_launch")

    def set_step_candidates(self, n_cand: int):
        """Decode steps rank blocks [0, n_cand) only (the complete blocks of a growing cache); 0 = all n_blocks."""
        self._check(self._L.sparda_set_step_candidates(self._h, int(n_cand)), "set_step_candidates")

    def set_step_selector(self, grid: bool, n_init: int = 0, n_local: int = 0):
        """grid=True: decode steps select with the (32,16) compressed-key grid (Kpool = Kgrid) and force init / local blocks."""
        self._check(self._L.sparda_set_step_selector(self._h, 1 if grid else 0, int(n_init), int(n_local)), "set_step_selector")

    def enable_peer_tier(self, peer_device: int):
        self._check(self._L.sparda_enable_peer_tier(self._h, int(peer_device)), "enable_peer_tier")

    def sparse_decode(self, Q, dev_pool, ids, topk, O, pool_is_indexed=False, n_slots=None, stream=None):
        n_slots = topk if n_slots is None else n_slots
        self._check(self._L.sparda_sparse_decode(self._h, _ptr(Q), _ptr(dev_pool), _ptr(ids), topk,
                                                 1 if pool_is_indexed else 0, n_slots, _ptr(O), _stream(stream)),
                    "sparse_decode")

    def sparse_decode_varlen(self, Q, dev_pool, ids, seq_len, topk, O, pool_is_indexed=False, n_slots=None, stream=None):
        n_slots = topk if n_slots is None else n_slots
        self._check(self._L.sparda_sparse_decode_varlen(self._h, _ptr(Q), _ptr(dev_pool), _ptr(ids), _ptr(seq_len), topk,
                                                        1 if pool_is_indexed else 0, n_slots, _ptr(O), _stream(stream)),
                    "sparse_decode_varlen")

    def make_layers(self, layers):
        """layers: list of dicts with tensors F, Q, Kpool, kv, O, ids -> ctypes array (keeps no references)."""
        arr = (SpardaLayer * len(layers))()
        for i, l in enumerate(layers):
            arr[i] = SpardaLayer(_ptr(l["F"]), _ptr(l["Q"]), _ptr(l["Kpool"]), _ptr(l["kv"]), _ptr(l["O"]), _ptr(l["ids"]),
                                 _ptr(l.get("X")) or None, _ptr(l.get("WF")) or None, _ptr(l.get("WFcur")) or None)
        return arr

    def decode_step(self, layer_array, F0cur, n_blocks, topk, pool0, pool1, compute_stream=None, prefetch_stream=None,
                    mode=STEP_OVERLAP):
        self._check(self._L.sparda_decode_step(self._h, layer_array, len(layer_array), _ptr(F0cur), n_blocks, topk,
                                               _ptr(pool0), _ptr(pool1), _stream(compute_stream),
                                               _stream(prefetch_stream), mode), "decode_step")

    def decode_step_host(self, layer_array, F0cur, n_blocks, topk, pool0, pool1, compute_stream=None,
                         prefetch_stream=None, mode=STEP_OVERLAP):
        """F, Q, O of every layer and F0cur are (pinned) HOST tensors; copies are enqueued inside the call."""
        self._check(self._L.sparda_decode_step_host(self._h, layer_array, len(layer_array), _ptr(F0cur), n_blocks, topk,
                                                    _ptr(pool0), _ptr(pool1), _stream(compute_stream),
                                                    _stream(prefetch_stream), mode), "decode_step_host")

    def reuse_plan(self, ids_new, topk, slot_ids, fetch, n_fetch=None, stream=None):
        self._check(self._L.sparda_reuse_plan(self._h, _ptr(ids_new), topk, _ptr(slot_ids), _ptr(fetch),
                                              _ptr(n_fetch) if n_fetch is not None else None, _stream(stream)), "reuse_plan")

    def forecast_select_plan(self, F, Kpool, n_blocks, topk, ids_out, slot_ids, fetch, n_fetch=None, n_cand=None, stream=None):
        n_cand = n_blocks if n_cand is None else n_cand
        self._check(self._L.sparda_forecast_select_plan(self._h, _ptr(F), _ptr(Kpool), n_blocks, n_cand, topk, _ptr(ids_out),
                                                        _ptr(slot_ids), _ptr(fetch), _ptr(n_fetch) if n_fetch is not None else None,
                                                        _stream(stream)), "forecast_select_plan")

    def make_cached_layers(self, layers):
        """layers: list of dicts with tensors F, Q, Kpool, kv, O, ids and (layers >= 1) pool, slot_ids, fetch, n_fetch."""
        arr = (SpardaCachedLayer * len(layers))()
        for i, l in enumerate(layers):
            base = SpardaLayer(_ptr(l["F"]), _ptr(l["Q"]), _ptr(l["Kpool"]), _ptr(l["kv"]), _ptr(l["O"]), _ptr(l["ids"]),
                               _ptr(l.get("X")) or None, _ptr(l.get("WF")) or None, _ptr(l.get("WFcur")) or None)
            opt = [(_ptr(l[n]) if l.get(n) is not None else None) for n in ("pool", "slot_ids", "fetch", "n_fetch")]
            arr[i] = SpardaCachedLayer(base, *opt)
        return arr

    def decode_step_cached(self, layer_array, F0cur, n_blocks, topk, compute_stream=None, prefetch_stream=None,
                           mode=STEP_OVERLAP):
        self._check(self._L.sparda_decode_step_cached(self._h, layer_array, len(layer_array), _ptr(F0cur), n_blocks, topk,
                                                      _stream(compute_stream), _stream(prefetch_stream), mode),
                    "decode_step_cached")

    def profile_enable(self, on=True):
        self._check(self._L.sparda_profile_enable(self._h, 1 if on else 0), "profile_enable")

    def profile_read(self):
        """-> {"select": (ms, n), "gather": (ms, n), "attn": (ms, n)} of the last decode_step."""
        ms = (ctypes.c_double * 3)()
        n = (ctypes.c_int64 * 3)()
        self._check(self._L.sparda_profile_read(self._h, ms, n), "profile_read")
        return {k: (ms[i], int(n[i])) for i, k in enumerate(("select", "gather", "attn"))}

    def prefill_select(self, F, Kpool, T, n_blocks, row0, n_rows, topk, ids_out, stream=None):
        self._check(self._L.sparda_prefill_select(self._h, _ptr(F), _ptr(Kpool), T, n_blocks, row0, n_rows, topk,
                                                  _ptr(ids_out), _stream(stream)), "prefill_select")

    def prefill_select_baseline(self, Q, Kpool, T, n_blocks, row0, n_rows, topk, ids_out, stream=None):
        self._check(self._L.sparda_prefill_select_baseline(self._h, _ptr(Q), _ptr(Kpool), T, n_blocks, row0, n_rows, topk,
                                                           _ptr(ids_out), _stream(stream)), "prefill_select_baseline")

    # ---- measurement aids (not the method) ----
    def probe_launch(self, kind, buf=None, nbytes=0, stream=None):
        self._check(self._L.sparda_probe_launch(self._h, kind, _ptr(buf), int(nbytes), _stream(stream)), "probe_launch")

    def set_layer_standin(self, weights=None, nbytes=0):
        self._check(self._L.sparda_set_layer_standin(self._h, _ptr(weights), int(nbytes)), "set_layer_standin")

    # ---- introspection ----
    @property
    def launch_count(self) -> int:
        return int(self._L.sparda_launch_count(self._h))

    @property
    def tmap_encodes(self) -> int:
        return int(self._L.sparda_tmap_encodes(self._h))

    @property
    def select_cluster(self) -> int:
        """Cluster size (CTAs per row) of the last forecast_select launch."""
        return int(self._L.sparda_get_select_cluster(self._h))

    @property
    def attn_cluster(self) -> int:
        """CTAs per row reduced through DSMEM by the last sparse_decode launch; 0 = workspace + ticket reduction."""
        return int(self._L.sparda_get_attn_cluster(self._h))

    def attn_splits(self, topk) -> int:
        return int(self._L.sparda_get_attn_splits(self._h, topk))

    @property
    def gather_ctas(self) -> int:
        return int(self._L.sparda_get_gather_ctas(self._h))


NOALLOC_MAX_ROWS = 256          # SPARDA_NOALLOC_MAX_ROWS
NOALLOC_SCRATCH_BYTES = 512 * (16 * 128 * 4 + 2 * 16 * 4) + 256 * 4   # SPARDA_NOALLOC_SCRATCH_BYTES


def sparse_decode_noalloc(batch, n_q_heads, n_kv_heads, head_dim, Q, dev_pool, ids, topk, O, pool_is_indexed=False,
                          n_slots=None, stream=None):
    """sparda_sparse_decode_noalloc: block-sparse attention without a context, for callers that must not allocate device
    memory (an engine that owns all of HBM, a loop that cannot take cudaMalloc's synchronisation, a plug-in with no set-up
    hook).  The split-K workspace is a fixed array inside libsparda (NOALLOC_SCRATCH_BYTES per GPU, rows <= NOALLOC_MAX_ROWS),
    shared by every call on the device: calls that may overlap on the GPU race.  Marshalling only."""
    L = lib()
    n_slots = topk if n_slots is None else n_slots
    rc = L.sparda_sparse_decode_noalloc(int(batch), int(n_q_heads), int(n_kv_heads), int(head_dim), _ptr(Q), _ptr(dev_pool),
                                        _ptr(ids), int(topk), 1 if pool_is_indexed else 0, int(n_slots), _ptr(O), _stream(stream))
    if rc != 0:
        raise SpardaError(f"sparse_decode_noalloc: {L.sparda_strerror(rc).decode()} [{rc}]: {L.sparda_noalloc_last_error().decode()}")


def version() -> str:
    return lib().sparda_version().decode()
