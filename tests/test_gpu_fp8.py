"""fp8 (e4m3) library storage (R26) through the C ABI against the oracle's fp8 path:
the stored codes and scale bytes bit-exact (both sides decide the code from the same exactly scaled value), the cache
stitched from fp8 segments: V bit-exact, shifted K within 1 bf16 ulp, page tables as ever."""
import numpy as np
import pytest
import torch

import fcg_testlib as T
from oracle import fcg_oracle as O
from paper_2606_13097_b200 import synth

pytestmark = pytest.mark.gpu


def _lib(L, Hq, Hkv, D, P, rope_mode, seg_tokens, n_pages=256, host_tier_tokens=0, base=1e4):
    from paper_2606_13097_b200.binding import FcgLibrary
    lib = FcgLibrary(n_layers=L, n_q_heads=Hq, n_kv_heads=Hkv, head_dim=D, page_size=P, rope_mode=rope_mode, rope_base=base,
                     max_segments=8, max_tasks=4, max_task_tokens=2048, n_pages=n_pages, segment_tokens=seg_tokens,
                     host_tier_tokens=host_tier_tokens)
    orc = O.OracleLibrary(L, Hq, Hkv, D, page_size=P, rope_mode=rope_mode, rope_base=base, n_pages=n_pages, max_task_tokens=2048)
    return lib, orc


def _compare_stored(lib, orc, sid):
    kc, vc, ke, ve = [x.cpu().numpy() for x in lib.segment_read(sid)]
    torch.cuda.synchronize()
    sg = orc.segments[sid]
    assert np.array_equal(ke.astype(np.int32) - 127, sg.k_exp), "K scale exponents"
    assert np.array_equal(ve.astype(np.int32) - 127, sg.v_exp), "V scale exponents"
    bad = np.argwhere(kc != sg.k)
    assert bad.size == 0, f"{len(bad)} K codes differ, first at {bad[:3].tolist()}: gpu {kc[tuple(bad[0])]:#x} oracle {sg.k[tuple(bad[0])]:#x}"
    assert np.array_equal(vc, sg.v), "V codes"


@pytest.mark.parametrize("D", [128, 64, 256, 96, 80, 192, 16])
def test_quantised_codes_and_scales_are_bit_exact(D):
    L, Hq, Hkv, P = 2, 4, 2, 16
    lib, orc = _lib(L, Hq, Hkv, D, P, 1, 4000)
    rng = np.random.default_rng(D)
    n = 300
    k = O.f64_to_bf16(rng.standard_normal((L, Hkv, n, D)))
    v = O.f64_to_bf16(rng.standard_normal((L, Hkv, n, D)) * np.exp(rng.uniform(-30, 30, (L, Hkv, n, 1))))     # row scales over 26 decades
    # rows at the edges of the format: zero rows, subnormal rows, huge rows, amax exactly on / just above 448 * 2^e,
    # exact ties of the e4m3 grid, non-finite elements
    k[:, :, 0] = 0
    k[:, :, 1] = 0x8000
    k[:, :, 2] = np.asarray([0x0001, 0x0040, 0x807F, 0x0000] * (D // 4), np.uint16)
    k[:, :, 3] = np.asarray([0x7F7F, 0xFF7F, 0x7F00, 0x3F80] * (D // 4), np.uint16)
    k[:, :, 4, :4] = [0x4060, 0x3F80, 0x3F88, 0x3F98]          # amax 3.5 -> e = -7: 1.0625 and 1.1875 are ties of the grid
    k[:, :, 5, :4] = [0x4061, 0x3F80, 0x3F88, 0x3F98]          # amax just above -> e = -6
    k[:, :, 6, 5], k[:, :, 6, 9], k[:, :, 6, 11] = 0x7F80, 0xFF80, 0x7FC1
    k[:, :, 7] = 0x7F80                                        # nothing finite in the row
    k[:, :, 8, ::2] = 0x0080                                   # smallest normals among N(0,1): they vanish (code 0)
    for i in range(16):                                        # every power-of-two amax boundary neighbourhood
        k[:, :, 20 + i, 0] = 0x3F60 + i                        # 0.875 .. in steps of one bf16 ulp
        k[:, :, 20 + i, 1:] = 0x3C00
    kt, vt = synth.from_bits(k, "cuda"), synth.from_bits(v, "cuda")
    sid = lib.segment_register_fp8(kt, vt, 17)
    assert sid == orc.segment_register_fp8(k, v, 17)
    _compare_stored(lib, orc, sid)
    fmt, nbytes = lib.segment_storage(sid)
    assert fmt == 1 and nbytes <= 2 * (L * Hkv * n * D + L * Hkv * n) + 4 * 256
    # a strided source (a slice of a bigger tensor) quantises to the same codes
    big_k = torch.zeros((L, Hkv, n + 40, D), dtype=torch.bfloat16, device="cuda")
    big_v = torch.zeros_like(big_k)
    big_k[:, :, 8:8 + n], big_v[:, :, 8:8 + n] = kt, vt
    sid2 = lib.segment_register_fp8(big_k[:, :, 8:8 + n], big_v[:, :, 8:8 + n], 17)
    assert sid2 == orc.segment_register_fp8(k, v, 17)
    _compare_stored(lib, orc, sid2)
    lib.close()


@pytest.mark.parametrize("D,rope_mode,P", [(128, 1, 16), (64, 1, 8), (128, 2, 32), (128, 0, 16), (256, 1, 16), (256, 2, 8), (96, 1, 16), (192, 2, 8), (80, 1, 32)])
def test_stitch_from_fp8_segments_matches_the_oracle(D, rope_mode, P):
    L, Hq, Hkv = 3, 4, 2
    lib, orc = _lib(L, Hq, Hkv, D, P, rope_mode, 6000, host_tier_tokens=600, base=5e5)
    rng = np.random.default_rng(7 * D + rope_mode)
    segs = []
    for i, (n, orig, fp8) in enumerate(((333, 1000, True), (150, 0, False), (500, 70, True), (64, 5, True))):
        k = O.f64_to_bf16(rng.standard_normal((L, Hkv, n, D)) * (1.0 if i != 3 else 1e-3))
        v = O.f64_to_bf16(rng.standard_normal((L, Hkv, n, D)) * (1.0 if i != 2 else 50.0))
        if fp8:
            sid = lib.segment_register_fp8(synth.from_bits(k, "cuda"), synth.from_bits(v, "cuda"), orig)
            assert sid == orc.segment_register_fp8(k, v, orig)
        else:
            sid = lib.segment_register(synth.from_bits(k, "cuda"), synth.from_bits(v, "cuda"), orig)
            assert sid == orc.segment_register(k, v, orig)
        segs.append(sid)
    lib.segment_offload(segs[2])                                # an offloaded fp8 segment is de-quantised straight from the host tier
    orc.segment_offload(segs[2])
    # fp8 and bf16 segments in one plan; sub-ranges; an identity graft (delta 0) of an fp8 segment; ragged page boundaries
    entries = [(segs[0], 5, 300, 0), (segs[1], 0, 150, 300), (segs[2], 17, 401, 455), (segs[3], 0, 64, 856), (segs[2], 0, 90, 920 + 70 - 70 + 0)]
    entries[4] = (segs[2], 0, 90, 990)
    plan_c = [{"task_id": 0, "entries": entries[:4], "holes": [(450, 5)], "capacity_tokens": 1000},
              {"task_id": 1, "entries": [(segs[2], 0, 500, 70), (segs[0], 0, 333, 600)], "holes": [], "capacity_tokens": 0}]
    plan_o = [O.Plan(0, [O.PlanEntry(*e) for e in entries[:4]], [O.Hole(450, 5)], 1000),
              O.Plan(1, [O.PlanEntry(segs[2], 0, 500, 70), O.PlanEntry(segs[0], 0, 333, 600)], [], 0)]
    lib.stitch(plan_c)
    orc.stitch(plan_o)
    assert orc.tasks[1].deltas[0] == 0                          # the identity graft: K is the de-quantised segment itself
    hist = np.zeros(4, np.int64)
    for tid in (0, 1):
        ot = orc.tasks[tid]
        assert np.array_equal(lib.task_page_table_host(tid), np.asarray(ot.page_table, np.int32))
        for layer in range(L):
            kg, vg = lib.task_read(tid, layer, 0, ot.capacity)
            f = ot.filled
            assert np.array_equal(synth.to_bits(vg)[:, f], ot.v[layer][:, f]), f"V from fp8 not bit-exact (task {tid} layer {layer})"
            hist += T.assert_k_within_1ulp(synth.to_bits(kg)[:, f], ot.k[layer][:, f], f"K from fp8, task {tid} layer {layer}")
    print(f"fp8 stitch D={D} rope_mode={rope_mode}: K ulp histogram [0,1,2,>=3] = {hist.tolist()}")
    kg, _ = lib.task_read(1, 0, 70, 500)
    sg = orc.segments[segs[2]]
    assert np.array_equal(synth.to_bits(kg), O.f64_to_bf16(O.fp8_dequantize_rows(sg.k[0], sg.k_exp[0])))
    # and a patch over a cache stitched from fp8 segments (the pages are bf16: attention is untouched)
    pos = np.arange(450, 455, dtype=np.int32)
    q = O.f64_to_bf16(rng.standard_normal((L, 5, Hq, D)))
    pk = O.f64_to_bf16(rng.standard_normal((L, 5, Hkv, D)))
    out = lib.patch(0, 0, synth.from_bits(q, "cuda"), synth.from_bits(pk, "cuda"), synth.from_bits(pk, "cuda"), pos)
    torch.cuda.synchronize()
    T.assert_attn_close(out, orc.patch(0, 0, q, pk, pk, pos), "patch over an fp8-stitched cache")
    lib.close()


def test_fp8_deep_subnormal_rows_and_special_codes_through_stitch():
    """scale clamped at 2^-127 (code * 2^e below bf16's range: one RNE), NaN codes, and -0"""
    L, Hq, Hkv, D, P = 1, 2, 1, 128, 16
    lib, orc = _lib(L, Hq, Hkv, D, P, 1, 200)
    n = 32
    k = np.zeros((L, Hkv, n, D), np.uint16)
    rng = np.random.default_rng(3)
    k[:] = rng.integers(0x0001, 0x0080, k.shape).astype(np.uint16)          # positive bf16 subnormals
    k[:, :, ::2] |= 0x8000
    k[:, :, 5, 3] = 0x7FC0
    k[:, :, 6] = O.f64_to_bf16(rng.standard_normal((L, Hkv, D)))
    k[:, :, 6, 40] = 0x7F80
    v = k[:, :, ::-1].copy()
    sid = lib.segment_register_fp8(synth.from_bits(k, "cuda"), synth.from_bits(v, "cuda"), 0)
    assert sid == orc.segment_register_fp8(k, v, 0)
    _compare_stored(lib, orc, sid)
    lib.stitch([{"task_id": 0, "entries": [(sid, 0, n, 0), (sid, 0, n, 40)], "holes": [(32, 8)], "capacity_tokens": 72}])
    orc.stitch([O.Plan(0, [O.PlanEntry(sid, 0, n, 0), O.PlanEntry(sid, 0, n, 40)], [O.Hole(32, 8)], 72)])
    kg, vg = lib.task_read(0, 0, 0, 72)
    f = orc.tasks[0].filled
    gk, gv, ok, ov = synth.to_bits(kg)[:, f], synth.to_bits(vg)[:, f], orc.tasks[0].k[0][:, f], orc.tasks[0].v[0][:, f]
    nan_o, nan_g = (ov & 0x7FFF) > 0x7F80, (gv & 0x7FFF) > 0x7F80
    assert np.array_equal(nan_o, nan_g) and np.array_equal(gv[~nan_o], ov[~nan_o])
    nan_o, nan_g = (ok & 0x7FFF) > 0x7F80, (gk & 0x7FFF) > 0x7F80
    assert np.array_equal(nan_o, nan_g)
    T.assert_k_within_1ulp(gk[~nan_o], ok[~nan_o], "deep subnormal K from fp8")
    lib.close()
