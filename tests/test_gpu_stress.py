"""`-m gpu` stress tests.  compute-sanitizer is closed on this pool, so races and stale reads are hunted with what is left:
random shapes against the oracle (every cluster size, ragged ranges, padded selections), NaN-poisoned pools that make
a missed or late copy visible, and repetition (the same inputs must give the same bits every time, eager or replayed
from a CUDA graph)."""
import numpy as np
import pytest
import torch

import parity
from paper_2606_04511_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sp():
    from paper_2606_04511_b200 import binding
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return binding


def _bits(t):
    return t.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16)


def test_select_random_shapes_against_oracle(sp, oracle):
    """120 random (D, Hkv, batch, n_blocks, k, n_cand, cluster size) selections, plain and fused with the reuse plan,
    checked against o3 + o4 (and o11 for the plan)."""
    rng = np.random.default_rng(2024)
    g = torch.Generator(device="cuda").manual_seed(2024)
    band = 0
    for it in range(120):
        D = int(rng.choice([64, 128]))
        Hkv = int(rng.integers(1, 4))
        B = int(rng.integers(1, 40))
        Nb = int(rng.integers(2, 1500)) if it % 10 else int(rng.integers(3000, 8193))
        k = int(rng.integers(1, min(256, Nb) + 1))
        cs = int(rng.choice([0, 0, 1, 2, 4, 8, 16]))
        cfg = synth.DecodeConfig("s", batch=B, n_q_heads=Hkv, n_kv_heads=Hkv, head_dim=D, n_blocks=Nb, topk=k)
        ctx = sp.Sparda.from_config(cfg, select_cluster=cs)
        R = cfg.rows
        kp = (torch.randn((R, Nb, D), generator=g, device="cuda") + torch.randn((R, Nb, 1), generator=g, device="cuda") * 1.5).to(torch.bfloat16)
        if it % 7 == 0:
            kp[:, Nb // 3] += 40.0                                    # a far positive outlier stretches the bucket range
        if it % 11 == 0:
            kp[:, : Nb // 2] = kp[:, Nb - Nb // 2:].clone()           # duplicated blocks: exact ties
        F = torch.randn((R, D), generator=g, device="cuda").to(torch.bfloat16)
        n_cand = int(rng.integers(0, Nb + 1)) if it % 3 else Nb
        ids = torch.full((R, k), -7, dtype=torch.int32, device="cuda")
        ctx.forecast_select(F, kp, Nb, k, ids, n_cand=n_cand)
        torch.cuda.synchronize()
        want, s = oracle.forecast_select(_bits(F), _bits(kp), k, n_cand)
        got = ids.cpu().numpy()
        band += parity.check_ids(got, want, s, n_cand)
        if it % 4 == 0:                                               # fused select + plan == select, then o11 on its ids
            slot = torch.from_numpy(rng.integers(-1, Nb, size=(R, k)).astype(np.int32)).cuda()
            old = slot.cpu().numpy().copy()
            ids2 = torch.full((R, k), -7, dtype=torch.int32, device="cuda")
            fetch = torch.full((R, k), -7, dtype=torch.int32, device="cuda")
            nf = torch.full((R,), -7, dtype=torch.int32, device="cuda")
            ctx.forecast_select_plan(F, kp, Nb, k, ids2, slot, fetch, nf, n_cand=n_cand)
            torch.cuda.synchronize()
            assert torch.equal(ids2, ids)
            want_after, want_fetch = oracle.reuse_plan(got, old)
            np.testing.assert_array_equal(slot.cpu().numpy(), want_after)
            np.testing.assert_array_equal(fetch.cpu().numpy(), want_fetch)
            np.testing.assert_array_equal(nf.cpu().numpy(), (want_fetch >= 0).sum(1))
        ctx.close()
    print(f"select stress: {band} rows used the near-tie band")


def _cached_layers(cfg, ctx, binding):
    R, k, Nb, D = cfg.rows, cfg.topk, cfg.n_blocks, cfg.head_dim
    dev = []
    for l in range(cfg.n_layers):
        L = synth.decode_layer(cfg, l, device="cuda")
        kpool = torch.empty((R, Nb, D), dtype=torch.bfloat16, device="cuda")
        ctx.pool_keys(L["kv"], R, Nb, kpool)
        dev.append({"F": L["F"].clone(), "F_base": L["F"], "Q": L["Q"], "Kpool": kpool, "kv": L["kv"] if l == 0 else L["kv"].cpu().pin_memory(),
                    "kv_bits": _bits(L["kv"]),
                    "O": torch.zeros((cfg.batch, cfg.n_q_heads, D), dtype=torch.bfloat16, device="cuda"),
                    "ids": torch.full((R, k), -9, dtype=torch.int32, device="cuda"),
                    "pool": torch.full((R, k, 2, 64, D), float("nan"), dtype=torch.bfloat16, device="cuda") if l else None,
                    "slot_ids": torch.full((R, k), -1, dtype=torch.int32, device="cuda") if l else None,
                    "fetch": torch.full((R, k), -9, dtype=torch.int32, device="cuda") if l else None,
                    "n_fetch": torch.zeros((R,), dtype=torch.int32, device="cuda") if l else None})
        if l == 0:
            F0 = L["F0cur"]
    return dev, F0


def test_cached_pipeline_is_deterministic_under_repetition(sp, oracle):
    """25 fresh runs of five drifting cached decode steps (6 layers, three streams, NaN-poisoned pools): every run gives
    the bits of the first, no NaN ever reaches O, and the first run's last step matches the oracle's attention over the
    pool the slot tables describe."""
    cfg = synth.DecodeConfig("p", batch=4, n_q_heads=32, n_kv_heads=2, head_dim=128, n_blocks=256, topk=64, n_layers=6, seed=5)
    ctx = sp.Sparda.from_config(cfg, max_layers=8)
    R, k, Nb, D = cfg.rows, cfg.topk, cfg.n_blocks, cfg.head_dim
    cs, ps = torch.cuda.Stream(), torch.cuda.Stream(priority=-1)
    ref = None
    for rep in range(25):
        dev, F0 = _cached_layers(cfg, ctx, sp)
        arr = ctx.make_cached_layers(dev)
        g = torch.Generator(device="cuda").manual_seed(1)
        outs = []
        for t in range(5):
            for d in dev:
                d["F"].copy_((d["F"].float() + 0.3 * torch.randn(d["F"].shape, generator=g, device="cuda")).to(torch.bfloat16))
            torch.cuda.synchronize()
            ctx.decode_step_cached(arr, F0, Nb, k, cs, ps, sp.STEP_OVERLAP)
            torch.cuda.synchronize()
            outs.append(torch.cat([d["O"].view(torch.int16).flatten() for d in dev] + [d["ids"].view(torch.int16).flatten() for d in dev]).clone())
        outs = torch.stack(outs)
        assert not torch.isnan(torch.stack([d["O"].float() for d in dev])).any(), f"rep {rep}: NaN reached O (a slot was read before it was filled)"
        if ref is None:
            ref = outs
            for l in range(1, cfg.n_layers):
                slots = dev[l]["slot_ids"].cpu().numpy()
                pool_ref = oracle.gather(dev[l]["kv_bits"], slots)
                got_pool = _bits(dev[l]["pool"])
                assert got_pool[slots >= 0].tobytes() == pool_ref[slots >= 0].tobytes()
                want, _ = oracle.sparse_attn(_bits(dev[l]["Q"]), pool_ref, slots)
                parity.check_attn(_bits(dev[l]["O"]), want, f"layer {l}")
        else:
            assert torch.equal(ref, outs), f"run {rep} differs from run 0"


def test_captured_cached_step_replays_with_poisoned_pools(sp, oracle):
    """One cached decode step captured into a CUDA graph (three streams, events, PDL edges) and replayed 30 times; before
    every replay the slot tables are reset and the pools poisoned with NaN, so that every replay must fetch everything
    again: O, ids, slot tables and pool bytes equal the eager step's every time, and the eager step matches the oracle."""
    cfg = synth.DecodeConfig("g", batch=3, n_q_heads=32, n_kv_heads=2, head_dim=128, n_blocks=300, topk=64, n_layers=5, seed=6)
    ctx = sp.Sparda.from_config(cfg, max_layers=8)
    R, k, Nb, D = cfg.rows, cfg.topk, cfg.n_blocks, cfg.head_dim
    dev, F0 = _cached_layers(cfg, ctx, sp)
    arr = ctx.make_cached_layers(dev)
    cs, ps = torch.cuda.Stream(), torch.cuda.Stream(priority=-1)

    def reset():
        for d in dev:
            d["O"].zero_()
            d["ids"].fill_(-9)
            if d["pool"] is not None:
                d["pool"].fill_(float("nan"))
                d["slot_ids"].fill_(-1)
                d["fetch"].fill_(-9)
        torch.cuda.synchronize()

    reset()
    ctx.decode_step_cached(arr, F0, Nb, k, cs, ps, sp.STEP_OVERLAP)
    torch.cuda.synchronize()
    names = ("O", "ids", "pool", "slot_ids", "fetch")
    want = [{n: d[n].clone() for n in names if d[n] is not None} for d in dev]
    for l, d in enumerate(dev):
        f = _bits(F0) if l == 0 else _bits(dev[l - 1]["F"])
        wi, s = oracle.forecast_select(f, _bits(d["Kpool"]), k)
        gids = d["ids"].cpu().numpy()
        parity.check_ids(gids, wi, s)
        if l == 0:
            wo, _ = oracle.sparse_attn(_bits(d["Q"]), d["kv_bits"], gids, pool_is_indexed=True)
        else:
            assert _bits(d["pool"]).tobytes() == oracle.gather(d["kv_bits"], d["slot_ids"].cpu().numpy()).tobytes()
            wo, _ = oracle.sparse_attn(_bits(d["Q"]), _bits(d["pool"]), d["slot_ids"].cpu().numpy())
        parity.check_attn(_bits(d["O"]), wo, f"layer {l}")
    graph = torch.cuda.CUDAGraph()
    reset()
    with torch.cuda.graph(graph, stream=cs):
        ctx.decode_step_cached(arr, F0, Nb, k, cs, ps, sp.STEP_OVERLAP)
    for rep in range(30):
        reset()
        graph.replay()
        torch.cuda.synchronize()
        for l, d in enumerate(dev):
            for n, wv in want[l].items():
                a, b = d[n], wv
                if a.dtype == torch.bfloat16:
                    a, b = a.view(torch.int16), b.view(torch.int16)
                assert torch.equal(a, b), f"replay {rep} layer {l} {n}"


def test_prefill_select_random_chunks_against_oracle(sp, oracle):
    """40 random chunk calls of the prefill selection (both tile modes, D, groups, k, ragged row ranges, several tiles per CTA),
    with planted ties: duplicated pooled keys, rows of all-equal scores, few distinct score values (the exact bitwise
    search), against o8.  The replicated mode re-arms its shared-memory exchange cells from tile to tile: every call here
    runs more than one tile per CTA at least in one group."""
    rng = np.random.default_rng(77)
    g = torch.Generator(device="cuda").manual_seed(77)
    band = rows = 0
    for it in range(40):
        D = int(rng.choice([64, 128]))
        Hkv = int(rng.integers(1, 4))
        Nb = int(rng.integers(3, 513))
        T = Nb * 64 + int(rng.integers(0, 64))
        k = int(rng.integers(1, min(64, Nb) + 1))
        ctx = sp.Sparda(1, Hkv, Hkv, D, Nb, k)
        kp = (torch.randn((Hkv, Nb, D), generator=g, device="cuda") + torch.randn((Hkv, Nb, 1), generator=g, device="cuda") * 1.5).to(torch.bfloat16)
        F = torch.randn((Hkv, T, D), generator=g, device="cuda").to(torch.bfloat16)
        n = int(rng.integers(1, min(T, 12000 if it % 8 == 0 else 3000) + 1))      # every 8th call is large enough for the 128-row tiles
        row0 = int(rng.integers(0, T - n + 1))
        if it % 3 == 0:
            kp[:, Nb // 2:] = kp[:, : Nb - Nb // 2].clone()               # duplicated keys: exact ties, lower id first
        if it % 4 == 0:
            F[:, row0 + n // 2: row0 + n // 2 + 40] = 0                   # all scores equal
        if it % 5 == 0:
            F[0, row0: row0 + 64, 1:] = 0                                 # scores = F[.,0] * Kpool[j,0] with few distinct values
            kp[0, :, 0] = (torch.arange(Nb, device="cuda") % 5).to(torch.bfloat16)
        ids = torch.full((Hkv, n, k), -7, dtype=torch.int32, device="cuda")
        ctx.prefill_select(F, kp, T, Nb, row0, n, k, ids)
        torch.cuda.synchronize()
        got = ids.cpu().numpy()
        # the oracle on sampled windows of the chunk (its cost grows with T * Nb): the head, the tail, the tie rows
        wins = {(0, min(n, 96)), (max(0, n - 96), min(n, 96)), (max(0, n // 2 - 8), min(n - max(0, n // 2 - 8), 64))}
        for w0, wn in wins:
            want, s = oracle.prefill_select(_bits(F), _bits(kp), k, row0 + w0, wn, want_scores=True)
            for gi in range(Hkv):
                ncand = np.minimum(Nb, (row0 + w0 + np.arange(wn) + 1) // 64)
                band += parity.check_ids(got[gi, w0:w0 + wn], want[gi], s[gi], ncand)
            rows += Hkv * wn
        valid = got >= 0
        ncand = np.minimum(Nb, (row0 + np.arange(n) + 1) // 64)
        assert np.array_equal(valid.sum(-1), np.broadcast_to(np.minimum(ncand, k), (Hkv, n))), f"case {it}: wrong id count"
        ctx.close()
    print(f"prefill stress: {band} of {rows} checked rows used the near-tie band")
