"""sparda_sparse_decode_noalloc: the block-sparse attention for callers that must not allocate device memory.

Who cannot allocate: a serving engine that gave all of HBM to its own pool at start-up (a library's cudaMalloc then
fails or eats into memory the engine thinks it owns), a decode loop that cannot take the device-wide synchronisation
cudaMalloc / cudaFree bring, a plug-in that only ever sees pointers and a stream.  None of them can go through
sparda_create, so this entry point takes no context and keeps its split-K workspace in one fixed array inside
libsparda (about 4.1 MiB per GPU, at most 256 rows = batch * n_kv_heads).

The GPU test checks it against the existing path (a context + sparda_sparse_decode) on several calls in a row on one
stream with no synchronisation between them, in the tolerances every attention test here uses (tests/parity.py), and
bit for bit where both sides are known to take the same split.  Every call shares the one array, so the calls of this
file stay on one stream.  The file is named to be collected last: `pytest -x` stops at the first failure, and a failure
here must not hide the parity tests.  It passes alone in a fresh process (the first call on the device does the
set-up) and after the other tests."""

import numpy as np
import pytest
import torch

import parity
from paper_2606_04511_b200 import synth

ELIMIT, EINVAL = -5, -1

# shapes: every one sends row partials through the scratch array
A4 = synth.DecodeConfig("na_r32_k64", batch=4, n_q_heads=32, n_kv_heads=8, head_dim=128, n_blocks=96, topk=64, seed=71)     # 4 CTAs per row
RAG = synth.DecodeConfig("na_ragged_k37", batch=3, n_q_heads=16, n_kv_heads=2, head_dim=128, n_blocks=300, topk=37, seed=72)  # CTA ranges cut rows anywhere
D64 = synth.DecodeConfig("na_d64_k19", batch=2, n_q_heads=8, n_kv_heads=2, head_dim=64, n_blocks=517, topk=19, seed=73)
MAXR = synth.DecodeConfig("na_256_rows", batch=32, n_q_heads=8, n_kv_heads=8, head_dim=64, n_blocks=16, topk=8, seed=74)     # the row limit: 2 partial slots per row


def _bits(t):
    return t.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16)


def test_noalloc_limits_are_refused_before_any_cuda_call():
    """Sizes beyond the fixed array come back as SPARDA_ELIMIT with a text that names the limit; the check runs before
    the first CUDA call, so it can be exercised without a GPU (the pointers are never dereferenced)."""
    from paper_2606_04511_b200 import binding, build
    build.build()
    L = binding.lib()
    fake = 0x10000   # aligned, never touched
    rc = L.sparda_sparse_decode_noalloc(33, 8, 8, 128, fake, fake, fake, 8, 0, 8, fake, None)    # 264 rows
    assert rc == ELIMIT
    msg = L.sparda_noalloc_last_error().decode()
    assert "264 rows" in msg and "SPARDA_NOALLOC_MAX_ROWS = 256" in msg, msg
    assert b"no-allocation" in L.sparda_strerror(ELIMIT)
    assert L.sparda_sparse_decode_noalloc(1, 8, 8, 96, fake, fake, fake, 8, 0, 8, fake, None) == EINVAL      # head_dim
    assert b"head_dim" in L.sparda_noalloc_last_error()
    assert L.sparda_sparse_decode_noalloc(1, 8, 8, 128, fake, fake, fake, 8, 0, 9, fake, None) == EINVAL     # n_slots != topk
    assert L.sparda_sparse_decode_noalloc(1, 8, 8, 128, fake, 0, fake, 8, 0, 8, fake, None) == EINVAL        # null pool
    with pytest.raises(binding.SpardaError, match="264 rows"):
        binding.sparse_decode_noalloc(33, 8, 8, 128, fake, fake, fake, 8, fake, stream=0)
    assert binding.NOALLOC_SCRATCH_BYTES == 4260864 and binding.NOALLOC_MAX_ROWS == 256


def _case(cfg, sp):
    """Inputs + the existing path's answers for one shape: ids from the context's select (one padded row, one empty row),
    the gathered pool, O through sparda_sparse_decode in both pool forms."""
    L = synth.decode_layer(cfg, 0, device="cuda")
    ctx = sp.Sparda.from_config(cfg)
    kpool = torch.empty((cfg.rows, cfg.n_blocks, cfg.head_dim), dtype=torch.bfloat16, device="cuda")
    ctx.pool_keys(L["kv"], cfg.rows, cfg.n_blocks, kpool)
    ids = torch.empty((cfg.rows, cfg.topk), dtype=torch.int32, device="cuda")
    ctx.forecast_select(L["F"], kpool, cfg.n_blocks, cfg.topk, ids)
    torch.cuda.synchronize()
    ids_np = ids.cpu().numpy().copy()
    ids_np[-1, cfg.topk - cfg.topk // 3:] = -1       # padded row
    ids_np[1, :] = -1                                # empty row -> zeros
    ids = torch.from_numpy(ids_np).cuda()
    pool = torch.zeros((cfg.rows, cfg.topk, 2, cfg.block_size, cfg.head_dim), dtype=torch.bfloat16, device="cuda")
    ctx.prefetch_launch(L["kv"], cfg.n_blocks, ids, cfg.topk, pool)
    want = torch.full((cfg.batch, cfg.n_q_heads, cfg.head_dim), float("nan"), dtype=torch.bfloat16, device="cuda")
    ctx.sparse_decode(L["Q"], pool, ids, cfg.topk, want)
    torch.cuda.synchronize()
    same_split = ctx.attn_cluster == 0               # the context also reduced through its workspace
    ctx.close()
    return {"cfg": cfg, "Q": L["Q"], "kv": L["kv"], "pool": pool, "ids": ids, "want": want, "same_split": same_split}


@pytest.mark.gpu
def test_noalloc_matches_existing_path_on_calls_in_a_row():
    from paper_2606_04511_b200 import binding as sp
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    cases = [_case(c, sp) for c in (A4, RAG, D64, MAXR)]
    st = torch.cuda.Stream()
    outs = []
    with torch.cuda.stream(st):
        # two rounds over all shapes back to back, no synchronisation in between: each call finds the array as the previous
        # one (another shape, another row count) left it.  Round 0 reads the gathered pool, round 1 the cache by block id.
        for rnd in range(2):
            for c in cases:
                cfg = c["cfg"]
                O = torch.full_like(c["want"], float("nan"))
                if rnd == 0:
                    sp.sparse_decode_noalloc(cfg.batch, cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim, c["Q"], c["pool"], c["ids"],
                                             cfg.topk, O, stream=st)
                else:
                    sp.sparse_decode_noalloc(cfg.batch, cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim, c["Q"], c["kv"], c["ids"],
                                             cfg.topk, O, pool_is_indexed=True, n_slots=cfg.n_blocks, stream=st)
                outs.append((rnd, c, O))
    st.synchronize()
    torch.cuda.synchronize()
    for rnd, c, O in outs:
        cfg = c["cfg"]
        what = f"{cfg.name} call round {rnd}"
        parity.check_attn(_bits(O), _bits(c["want"]), what)
        b, g = divmod(1, cfg.n_kv_heads)
        assert torch.all(O[b, g * cfg.group:(g + 1) * cfg.group] == 0), f"{what}: an empty row must give O = 0"
        if c["same_split"]:
            assert torch.equal(O.view(torch.int16), c["want"].view(torch.int16)), f"{what}: same split as the context, bits differ"
    assert any(c["same_split"] for c in cases)
