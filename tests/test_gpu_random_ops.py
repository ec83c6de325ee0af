"""Randomised differential test: seeded sequences of library operations (register, stitch, patch, decode, shift,
extract, offload / prefetch, release) run on the CUDA library and on the oracle side by side; after every step the
page tables, pool / segment bookkeeping and every filled cache position are compared (V bits, K within 1 ulp --
or bit-exact where no rotation happened since the last comparison -- attention within tolerance).  Small
geometries, many steps: aimed at the state machine (allocate-then-commit, page recycling, fill tracking)."""
import numpy as np
import pytest
import torch

from oracle import fcg_oracle as O
from paper_2606_13097_b200 import synth
import fcg_testlib as T

pytestmark = pytest.mark.gpu


def _pair_close(a_bits, b_bits, c, rope_mode):
    """|a - b| <= c * 2^-9 * |rotation pair| per component"""
    a, b = O.bf16_to_f64(a_bits), O.bf16_to_f64(b_bits)
    if rope_mode == 2:
        norm = np.repeat(np.sqrt(b[..., 0::2] ** 2 + b[..., 1::2] ** 2), 2, axis=-1)
    else:
        half = b.shape[-1] // 2
        n = np.sqrt(b[..., :half] ** 2 + b[..., half:] ** 2)
        norm = np.concatenate([n, n], axis=-1)
    return bool(np.all(np.abs(a - b) <= c * 2.0 ** -9 * norm + 1e-30))


def _pick_range(rng, ot, n_max):
    """mostly a sub-range of a filled run of the task (so the call is accepted), sometimes anything (rejections)"""
    f = ot.filled
    if rng.random() < 0.25 or not f.any():
        return int(rng.integers(0, ot.capacity)), int(rng.integers(1, n_max))
    edges = np.flatnonzero(np.diff(np.concatenate([[0], f.astype(np.int8), [0]])))
    runs = list(zip(edges[0::2], edges[1::2]))
    b0, e0 = runs[int(rng.integers(len(runs)))]
    b = int(rng.integers(b0, e0))
    return b, int(rng.integers(1, min(n_max, e0 - b) + 1))


def _bits(rng, shape):
    x = torch.from_numpy(rng.standard_normal(shape).astype(np.float32)).to(torch.bfloat16)
    return x, synth.to_bits(x)


@pytest.mark.parametrize("seed,D,Hq,Hkv,P,rope_mode", [(11, 128, 4, 2, 16, 1), (12, 64, 4, 4, 8, 1), (13, 128, 8, 2, 32, 2),
                                                     (14, 128, 2, 1, 16, 0), (15, 128, 6, 2, 64, 1), (16, 256, 4, 2, 16, 1), (17, 96, 4, 2, 16, 1), (18, 160, 4, 4, 32, 2)])
def test_random_operation_sequences(seed, D, Hq, Hkv, P, rope_mode):
    from paper_2606_13097_b200.binding import FcgLibrary, FcgError
    rng = np.random.default_rng(seed)
    L, max_tasks, max_segments, cap_max, n_pages = 2, 3, 6, 320, 3 * (320 // P) + 7
    lib = FcgLibrary(n_layers=L, n_q_heads=Hq, n_kv_heads=Hkv, head_dim=D, page_size=P, rope_mode=rope_mode, rope_base=1e4,
                     max_segments=max_segments, max_tasks=max_tasks, max_task_tokens=cap_max, n_pages=n_pages,
                     segment_tokens=2000, host_tier_tokens=1200)
    orc = O.OracleLibrary(L, Hq, Hkv, D, page_size=P, rope_mode=rope_mode, rope_base=1e4, max_segments=max_segments,
                          max_tasks=max_tasks, n_pages=n_pages, max_task_tokens=cap_max)
    seg_tokens_dev = 0          # arena accounting the oracle does not model: stay far below capacity (fragmentation)
    seg_gen, task_gen = {}, {}  # re-rotation generations of the K data (see compare_all)

    def both(name, *args):
        """run the same call on both sides; statuses must agree; returns (gpu result, oracle result) or None on a rejection"""
        try:
            ro = getattr(orc, name)(*args)
            err_o = None
        except O.OracleError as e:
            ro, err_o = None, e.status
        try:
            rg = getattr(lib, name)(*args)
            err_g = None
        except FcgError as e:
            rg, err_g = None, e.status
        assert err_o == err_g, f"{name}{args}: oracle status {err_o}, library status {err_g}"
        return None if err_o is not None else (rg, ro)

    def compare_all():
        assert lib.pool_info()["n_pages_free"] == orc.pool.available()
        assert lib.pool_info()["n_tasks_live"] == len(orc.tasks) and lib.pool_info()["n_segments_live"] == len(orc.segments)
        for tid, ot in orc.tasks.items():
            assert np.array_equal(lib.task_page_table_host(tid), np.asarray(ot.page_table, np.int32)), f"task {tid} page table"
            assert lib.task_page_table(tid)[2] == ot.n_tokens
            for layer in range(L):
                k, v = lib.task_read(tid, layer, 0, ot.capacity)
                kb, vb = synth.to_bits(k), synth.to_bits(v)
                f = ot.filled
                assert np.array_equal(vb[:, f], ot.v[layer][:, f]), f"task {tid} layer {layer}: V"
                if rope_mode == 0 or task_gen[tid] == 0:
                    T.assert_k_within_1ulp(kb[:, f], ot.k[layer][:, f], f"task {tid} layer {layer}")
                else:
                    # data that went through g earlier shift / extract generations: each generation both sides round
                    # once, from inputs that may already differ by a rounding -- bound relative to the pair norm
                    assert _pair_close(kb[:, f], ot.k[layer][:, f], 2.5 * (task_gen[tid] + 1), rope_mode), \
                        f"task {tid} layer {layer}: K after {task_gen[tid]} re-rotation generation(s)"
        for sid, sg in orc.segments.items():
            assert lib.segment_info(sid) == (sg.n_tokens, sg.orig_start, sg.resident)

    n_ops = {"stitch": 0, "patch": 0, "shift": 0, "extract": 0, "tier": 0, "rejected": 0}
    for step in range(120):
        op = rng.choice(["register", "stitch", "patch", "decode", "shift", "extract", "tier", "release_task", "release_seg"],
                        p=[0.14, 0.16, 0.14, 0.12, 0.14, 0.08, 0.1, 0.07, 0.05])
        live_t, live_s = sorted(orc.tasks), sorted(orc.segments)
        if op == "register" and len(live_s) < max_segments:
            n = int(rng.integers(5, 120))
            if seg_tokens_dev + n > 800:
                continue
            (kt, kb), (vt, vb) = _bits(rng, (L, Hkv, n, D)), _bits(rng, (L, Hkv, n, D))
            start = int(rng.integers(0, 5000))
            sid = orc.segment_register(kb, vb, start)
            assert lib.segment_register(kt.cuda(), vt.cuda(), start) == sid
            seg_gen[sid] = 0
            seg_tokens_dev += n
        elif op == "stitch" and live_s and len(live_t) < max_tasks:
            tid = next(t for t in range(max_tasks) if t not in orc.tasks)
            entries, holes, cursor = [], [], 0
            for _ in range(int(rng.integers(1, 4))):
                s = int(rng.choice(live_s))
                ns = orc.segments[s].n_tokens
                b = int(rng.integers(0, ns))
                n = int(rng.integers(1, ns - b + 1))
                if rng.random() < 0.3:
                    h = int(rng.integers(1, 20))
                    holes.append((cursor, h))
                    cursor += h
                entries.append((s, b, n, cursor))
                cursor += n
            cap = cursor + int(rng.integers(0, 40))
            if rng.random() < 0.1:
                entries.append(entries[0])                        # overlap -> both must reject
            try:
                orc.stitch([O.Plan(tid, [O.PlanEntry(*e) for e in entries], [O.Hole(*h) for h in holes], cap)])
                eo = None
            except O.OracleError as e:
                eo = e.status
            try:
                lib.stitch([{"task_id": tid, "entries": entries, "holes": holes, "capacity_tokens": cap}])
                eg = None
            except FcgError as e:
                eg = e.status
            assert eo == eg, f"stitch: oracle {eo}, library {eg}"
            n_ops["stitch" if eo is None else "rejected"] += 1
            if eo is None:
                task_gen[tid] = max(seg_gen[e[0]] for e in entries)
        elif op in ("patch", "decode") and live_t:
            tid = int(rng.choice(live_t))
            ot = orc.tasks[tid]
            unfilled = np.flatnonzero(~ot.filled)
            if op == "patch" and unfilled.size:
                first = int(unfilled[0])
                run = 1
                while first + run < ot.capacity and not ot.filled[first + run] and run < 24:
                    run += 1
                pos = np.arange(first, first + run, dtype=np.int32)
                if first > 0 and not ot.filled[:first].all():
                    pos = pos[:1]
            else:
                filled = np.flatnonzero(ot.filled)
                if filled.size == 0:
                    continue
                pos = np.asarray([int(rng.choice(filled))], np.int32)     # re-patch (decode-like) of a filled position
            (qt, qb), (kt, kb), (vt, vb) = _bits(rng, (L, len(pos), Hq, D)), _bits(rng, (L, len(pos), Hkv, D)), _bits(rng, (L, len(pos), Hkv, D))
            try:
                ref = orc.patch(tid, 0, qb, kb, vb, pos)
                eo = None
            except O.OracleError as e:
                eo = e.status
            try:
                out = lib.patch(tid, 0, qt.cuda(), kt.cuda(), vt.cuda(), pos)
                eg = None
            except FcgError as e:
                eg = e.status
            assert eo == eg, f"patch at {pos.tolist()}: oracle {eo}, library {eg}"
            if eo is None:
                T.assert_attn_close(out, ref, f"step {step} patch task {tid} positions {pos.tolist()}")
                n_ops["patch"] += 1
            else:
                n_ops["rejected"] += 1
        elif op == "shift" and live_t:
            tid = int(rng.choice(live_t))
            ot = orc.tasks[tid]
            src, n = _pick_range(rng, ot, 60)
            dst = max(0, src + int(rng.integers(-40, 41)))
            r = both("task_shift", tid, src, n, dst)
            n_ops["shift" if r is not None else "rejected"] += 1
            if r is not None and dst != src:
                task_gen[tid] += 1
        elif op == "extract" and live_t and len(live_s) < max_segments:
            tid = int(rng.choice(live_t))
            ot = orc.tasks[tid]
            b, n = _pick_range(rng, ot, 50)
            if seg_tokens_dev + n > 800:
                continue
            r = both("segment_extract", tid, b, n, int(rng.choice([0, b, 77])))
            if r is not None:
                assert r[0] == r[1]
                seg_gen[r[1]] = task_gen[tid] + 1
                seg_tokens_dev += n
                n_ops["extract"] += 1
            else:
                n_ops["rejected"] += 1
        elif op == "tier" and live_s:
            s = int(rng.choice(live_s))
            sg = orc.segments[s]
            if sg.resident:
                both("segment_offload", s)
                seg_tokens_dev -= sg.n_tokens
            elif seg_tokens_dev + sg.n_tokens <= 800:
                both("segment_prefetch", s)
                seg_tokens_dev += sg.n_tokens
            n_ops["tier"] += 1
        elif op == "release_task" and live_t:
            both("task_release", int(rng.choice(live_t)))
        elif op == "release_seg" and live_s:
            s = int(rng.choice(live_s))
            if orc.segments[s].resident:
                seg_tokens_dev -= orc.segments[s].n_tokens
            both("segment_release", s)
        else:
            continue
        torch.cuda.synchronize()
        compare_all()
    print(f"seed {seed}: {n_ops}")
    assert n_ops["stitch"] >= 3 and n_ops["patch"] + n_ops["shift"] >= 3
    lib.close()
