"""Out-of-bounds and uninitialised-read checks of our own.  compute-sanitizer is closed on this GPU pool (gpurun answers
"compute-sanitizer is closed on this pool and stays closed"; profiles/r02_sanitizer.md), so the sanitizer tier of
SURVEY.md 4 / 5 is replaced by what can be checked from outside the kernels:

* memcheck substitute: the library's arena and every caller buffer (q, k, v, out, segment sources, read-back targets)
  sit inside larger allocations filled with a canary byte; after a sequence that goes through every kernel of the
  library (both attention paths, split-KV + combine, fp8, shift, extract, host and rope variants, plans) every guard
  zone must still hold the canary;
* initcheck substitute: the page pool and the workspace are poisoned with NaN patterns before use and `out` is
  pre-filled with NaN: results must match the oracle and hold no NaN, i.e. nothing that was never written is read
  and every output row is written.
"""
import numpy as np
import pytest
import torch

import fcg_testlib as T
from oracle import fcg_oracle as O
from paper_2606_13097_b200 import synth

pytestmark = pytest.mark.gpu
CANARY = 0xA5
GUARD = 1 << 20


class Guarded:
    """a tensor view in the middle of a canary-filled allocation"""

    def __init__(self, shape, dtype, fill=None):
        nbytes = int(np.prod(shape)) * torch.empty((), dtype=dtype).element_size()
        self.raw = torch.full((nbytes + 2 * GUARD,), CANARY, dtype=torch.uint8, device="cuda")
        self.view = self.raw[GUARD:GUARD + nbytes].view(dtype).view(*shape)
        self.nbytes = nbytes
        if fill is not None:
            self.view.copy_(fill)

    def intact(self):
        lo, hi = self.raw[:GUARD], self.raw[GUARD + self.nbytes:]
        return bool((lo == CANARY).all()) and bool((hi == CANARY).all())


def _guarded_library(L, Hq, Hkv, D, P, rope_mode, seg_tokens, n_pages, max_task_tokens, workspace=64 << 20):
    from paper_2606_13097_b200 import binding as B
    cfg = B.make_config(n_layers=L, n_q_heads=Hq, n_kv_heads=Hkv, head_dim=D, page_size=P, rope_mode=rope_mode, rope_base=1e4,
                        max_segments=8, max_tasks=3, max_task_tokens=max_task_tokens, n_pages=n_pages, workspace_bytes=workspace)
    need = B.fcg_arena_bytes_required(cfg, seg_tokens)
    g = Guarded((need,), torch.uint8)
    g.view.view(torch.int16).fill_(0x7FC1)                       # poison: every never-written byte of the arena is a NaN pattern
    cfg.arena, cfg.arena_bytes = g.view.data_ptr(), need
    lib = B.FcgLibrary.__new__(B.FcgLibrary)
    lib.n_layers, lib.n_q_heads, lib.n_kv_heads, lib.head_dim, lib.page_size = L, Hq, Hkv, D, P
    lib.device, lib.host_arena, lib.arena = torch.device("cuda", 0), None, g.view
    lib.handle = B.fcg_library_create(cfg)
    return lib, g


@pytest.mark.parametrize("D,rope_mode", [(128, 1), (64, 2), (256, 1), (96, 1), (176, 2)])
def test_no_kernel_writes_outside_its_buffers_and_nothing_unwritten_is_read(D, rope_mode):
    L, Hq, Hkv, P = 3, 8, 2, 16
    rng = np.random.default_rng(D)
    lib, g_arena = _guarded_library(L, Hq, Hkv, D, P, rope_mode, 3000, 200, 1500)
    orc = O.OracleLibrary(L, Hq, Hkv, D, page_size=P, rope_mode=rope_mode, rope_base=1e4, n_pages=200, max_task_tokens=1500)
    guards = [g_arena]

    def dev(bits):
        g = Guarded(bits.shape, torch.bfloat16, synth.from_bits(bits, "cuda"))
        guards.append(g)
        return g.view

    def rnd(shape):
        return O.f64_to_bf16(rng.standard_normal(shape))

    segs = []
    for i, (n, fp8) in enumerate(((333, False), (700, False), (257, True))):
        k, v = rnd((L, Hkv, n, D)), rnd((L, Hkv, n, D))
        if fp8:
            sid = lib.segment_register_fp8(dev(k), dev(v), 40 * i)
            assert sid == orc.segment_register_fp8(k, v, 40 * i)
        else:
            sid = lib.segment_register(dev(k), dev(v), 40 * i)
            assert sid == orc.segment_register(k, v, 40 * i)
        segs.append(sid)
    entries = [(segs[0], 3, 300, 0), (segs[1], 0, 700, 317), (segs[2], 0, 257, 1017)]
    lib.stitch([{"task_id": 0, "entries": entries, "holes": [(300, 17)], "capacity_tokens": 1290}])
    orc.stitch([O.Plan(0, [O.PlanEntry(*e) for e in entries], [O.Hole(300, 17)], 1290)])

    def patch_both(fn_name, pos, layer_begin=0, n_layers=L, splits=0, tc_min_rows=1, raw_qk=False):
        n = len(pos)
        q, k, v = rnd((n_layers, n, Hq, D)), rnd((n_layers, n, Hkv, D)), rnd((n_layers, n, Hkv, D))
        lib.set_attn_policy(tc_min_rows, splits)
        out = Guarded((n_layers, n, Hq, D), torch.bfloat16)
        out.view.view(torch.int16).fill_(0x7FC1)                  # an output row that is never written stays NaN
        guards.append(out)
        ref = (orc.patch_rope if raw_qk else orc.patch)(0, layer_begin, q, k, v, pos)
        if fn_name == "host":
            qh, kh, vh = [synth.from_bits(x).pin_memory() for x in (q, k, v)]
            oh = torch.empty_like(qh).pin_memory()
            lib.patch_host(0, layer_begin, qh, kh, vh, pos, oh)
            torch.cuda.synchronize()
            out.view.copy_(oh)
        else:
            getattr(lib, fn_name)(0, layer_begin, dev(q), dev(k), dev(v), pos, out.view)
        torch.cuda.synchronize()
        assert not torch.isnan(out.view.float()).any(), f"{fn_name}: an output row was never written (or read poison)"
        T.assert_attn_close(out.view, ref, f"{fn_name} pos {pos[0]}..{pos[-1]} splits {splits} tc_min_rows {tc_min_rows}")

    mid = np.arange(300, 317, dtype=np.int32)
    patch_both("patch", mid)                                                 # tcgen05, one split
    patch_both("patch", mid, splits=3)                                       # tcgen05, split-KV partials + combine
    patch_both("patch", mid, splits=2, tc_min_rows=2 ** 31 - 1)              # mma.sync split-KV path + combine
    patch_both("patch", np.arange(1274, 1290, dtype=np.int32))
    patch_both("patch", mid, layer_begin=1, n_layers=2)                      # a layer sub-range (re-patch: positions stay filled in every layer)
    patch_both("patch", np.arange(1290, 1300, dtype=np.int32))               # append beyond the capacity (R25)
    patch_both("host", np.arange(1300, 1340, dtype=np.int32), splits=2)      # 160 rows per kv head: tile-parity / two-Q-tile classes
    patch_both("patch_rope", np.arange(1340, 1345, dtype=np.int32), raw_qk=True)
    plan = lib.patch_plan_create([0], [3], [1345, 1346, 1347], 1)
    q, k, v = rnd((L, 3, Hq, D)), rnd((L, 3, Hkv, D)), rnd((L, 3, Hkv, D))
    out = Guarded((L, 3, Hq, D), torch.bfloat16)
    guards.append(out)
    qd, kd, vd = dev(q), dev(k), dev(v)
    for layer in range(L):
        lib.patch_planned(plan, layer, qd[layer:layer + 1], kd[layer:layer + 1], vd[layer:layer + 1], out.view[layer:layer + 1])
    torch.cuda.synchronize()
    T.assert_attn_close(out.view, orc.patch(0, 0, q, k, v, [1345, 1346, 1347]), "planned per-layer calls")
    lib.patch_plan_destroy(plan)
    lib.task_shift(0, 400, 500, 420)
    orc.task_shift(0, 400, 500, 420)
    sid = lib.segment_extract(0, 0, 290, 0)
    assert sid == orc.segment_extract(0, 0, 290, 0)
    ot = orc.tasks[0]
    for layer in range(L):
        kg = Guarded((Hkv, ot.capacity, D), torch.bfloat16)
        vg = Guarded((Hkv, ot.capacity, D), torch.bfloat16)
        guards += [kg, vg]
        from paper_2606_13097_b200 import binding as B
        B.fcg_task_read(lib.handle, 0, layer, 0, ot.capacity, kg.view, vg.view)
        torch.cuda.synchronize()
        f = ot.filled
        assert np.array_equal(synth.to_bits(vg.view)[:, f], ot.v[layer][:, f])
        # the shifted range [420, 920) was rotated twice, each side from its own (<= 1 ulp apart) first result: bounded
        # relative to the rotation pair there (a ulp count says nothing about the small component of a pair)
        once = f.copy()
        once[420:920] = False
        T.assert_k_within_1ulp(synth.to_bits(kg.view)[:, once], ot.k[layer][:, once], f"layer {layer}")
        assert T.k_pair_close(synth.to_bits(kg.view)[:, 420:920], ot.k[layer][:, 420:920], 5.0, rope_mode), f"layer {layer}: twice-rotated keys"
    ks, vs = lib.segment_read(sid)
    torch.cuda.synchronize()
    assert np.array_equal(synth.to_bits(vs), orc.segments[sid].v)
    T.assert_k_within_1ulp(synth.to_bits(ks), orc.segments[sid].k, "extracted segment")
    bad = [i for i, g in enumerate(guards) if not g.intact()]
    assert not bad, f"guard zones of buffers {bad} were written (0 = the library arena)"
    lib.close()
