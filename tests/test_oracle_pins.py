"""Pins for the CPU oracle: the oracle is checked against things
other than itself -- golden closed forms, algebraic invariants, brute force in pure python
loops, independent formulas (complex multiplication, HF-style rotate_half in torch), and a
library routine (torch SDPA fp64).  CPU only.
"""
import cmath
import math
import os

import numpy as np
import pytest
import torch

from oracle import fcg_oracle as O

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
RNG = np.random.default_rng(20260613)


def _bf16_bits_from_f32(x32: np.ndarray) -> np.ndarray:
    """torch's fp32->bf16 RNE cast as an independent witness (valid when x is already an fp32 value)."""
    return torch.from_numpy(np.ascontiguousarray(x32, np.float32)).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)


def _rand_bf16(shape, scale=1.0):
    x = (RNG.standard_normal(shape) * scale).astype(np.float32)
    return _bf16_bits_from_f32(x)


def _ulp_dist(a_bits, b_bits):
    """distance in bf16 ulps via the monotone integer mapping of sign-magnitude floats."""
    def key(b):
        b = b.astype(np.int32)
        return np.where(b & 0x8000, 0x8000 - b, b)   # negative -> -(magnitude)
    return np.abs(key(np.asarray(a_bits)) - key(np.asarray(b_bits)))


# ----------------------------------------------------------------------------------------------
# bf16 conversion
# ----------------------------------------------------------------------------------------------
def test_bf16_rounding_golden():
    n = 0
    for line in open(os.path.join(GOLDEN, "bf16_rounding.txt")):
        if line.startswith("#") or not line.strip():
            continue
        expr, hexbits, _why = [p.strip() for p in line.split("|")]
        x = eval(expr, {"__builtins__": {}})
        got = int(O.f64_to_bf16(np.array([x]))[0])
        assert got == int(hexbits, 16), (expr, hex(got), hexbits)
        n += 1
    assert n >= 15


def test_bf16_roundtrip_all_patterns():
    """every finite bf16 pattern converts to fp64 and back to itself; matches torch's widening."""
    bits = np.arange(0x10000, dtype=np.uint32).astype(np.uint16)
    f = O.bf16_to_f64(bits)
    wide = torch.from_numpy(bits.view(np.int16)).view(torch.bfloat16).to(torch.float64).numpy()
    finite = np.isfinite(wide)
    assert np.array_equal(f[finite], wide[finite])
    back = O.f64_to_bf16(f)
    assert np.array_equal(back[finite], bits[finite])
    inf = np.isinf(wide)
    assert np.array_equal(back[inf], bits[inf])
    assert np.all(np.isnan(f[np.isnan(wide)]))


def test_bf16_rounding_matches_torch_on_fp32_inputs():
    """when the double IS an fp32 value there is no double rounding, so torch's cast must agree."""
    x32 = np.concatenate([RNG.standard_normal(200000).astype(np.float32) * 10.0 ** RNG.integers(-30, 30, 200000),
                          np.float32([0.0, -0.0, 1e-40, -1e-40, 3.3e38, 3.39e38, 3.4e38])]).astype(np.float32)
    assert np.array_equal(O.f64_to_bf16(x32.astype(np.float64)), _bf16_bits_from_f32(x32))


def test_bf16_rounding_is_nearest():
    """brute force: the result is the closest bf16 value (checked against both neighbours)."""
    x = RNG.standard_normal(20000) * 3.0
    b = O.f64_to_bf16(x)
    c = O.bf16_to_f64(b)
    lo = O.bf16_to_f64((b.astype(np.int32) - 1).astype(np.uint16))
    hi = O.bf16_to_f64((b.astype(np.int32) + 1).astype(np.uint16))
    err = np.abs(c - x)
    assert np.all(err <= np.abs(lo - x)) and np.all(err <= np.abs(hi - x))


# ----------------------------------------------------------------------------------------------
# RoPE: closed forms and invariants
# ----------------------------------------------------------------------------------------------
def test_inv_freq_definition():
    th = O.rope_inv_freq(8, 1e4)
    assert np.allclose(th, [1.0, 0.1, 0.01, 0.001], rtol=1e-15)
    th = O.rope_inv_freq(128, 5e5)
    assert th[0] == 1.0 and th.shape == (64,)
    assert math.isclose(th[32], 5e5 ** -0.5, rel_tol=1e-15)
    assert np.all(np.diff(th) < 0)


def test_rope_closed_forms_golden():
    n = 0
    for line in open(os.path.join(GOLDEN, "rope_closed_forms.txt")):
        if line.startswith("#") or not line.strip():
            continue
        head, kvals, exact, hexes = [p.split() for p in line.split("|")]
        D, base, delta = int(head[0]), float(head[1]), int(head[2])
        k = np.array([float(v) for v in kvals])
        want = np.array([float(v) for v in exact])
        got = O.rope_rotate_f64(k, delta, O.rope_inv_freq(D, base))
        # fp64 cos/sin of angles up to 3e4 rad carry ~|phi|*2^-53 absolute error
        assert np.allclose(got, want, rtol=0, atol=1e-11), (line, got)
        assert [f"{b:04X}" for b in O.f64_to_bf16(got)] == hexes
        # the bf16 path as the stitch uses it (inputs here are exactly representable in bf16)
        kb = O.f64_to_bf16(k)
        assert np.array_equal(O.bf16_to_f64(kb), k)
        assert [f"{b:04X}" for b in O.rope_shift_bf16(kb, delta, O.rope_inv_freq(D, base))] == hexes
        n += 1
    assert n >= 5


def test_rope_matches_complex_multiplication():
    """independent formula: (a + ib) * exp(i*delta*theta) -- catches sign / pairing / transposition errors."""
    D = 16
    th = O.rope_inv_freq(D, 1e4)
    k = RNG.standard_normal((5, D))
    for delta in (-300, -1, 0, 1, 77, 4095):
        got = O.rope_rotate_f64(k, delta, th)
        for r in range(5):
            for j in range(D // 2):
                z = complex(k[r, j], k[r, j + D // 2]) * cmath.exp(1j * delta * th[j])
                assert math.isclose(got[r, j], z.real, rel_tol=0, abs_tol=1e-12)
                assert math.isclose(got[r, j + D // 2], z.imag, rel_tol=0, abs_tol=1e-12)


def test_rope_matches_hf_rotate_half_restated():
    """The HF convention (the paper's stack): x*cos + rotate_half(x)*sin with
    rotate_half(x) = cat(-x2, x1) and cos/sin = cat(freqs, freqs); restated with torch fp64 ops."""
    D, delta = 32, 911
    k = torch.from_numpy(RNG.standard_normal((7, D)))
    inv = 1.0 / (1e4 ** (torch.arange(0, D, 2, dtype=torch.float64) / D))
    emb = torch.cat([delta * inv, delta * inv])
    rot = torch.cat([-k[:, D // 2:], k[:, : D // 2]], dim=-1)
    want = k * emb.cos() + rot * emb.sin()
    got = O.rope_rotate_f64(k.numpy(), delta, O.rope_inv_freq(D, 1e4))
    assert np.allclose(got, want.numpy(), rtol=0, atol=1e-12)


def test_p1_group_law():
    D = 64
    th = O.rope_inv_freq(D, 1e4)
    k = RNG.standard_normal((50, D))
    for a, b in ((3, 5), (-100, 40), (2048, -2048), (12345, 4321)):
        lhs = O.rope_rotate_f64(O.rope_rotate_f64(k, a, th), b, th)
        rhs = O.rope_rotate_f64(k, a + b, th)
        assert np.max(np.abs(lhs - rhs)) <= 1e-11
    # with a bf16 rounding in between: each pair within 2 bf16 ulp of the pair norm
    kb = _rand_bf16((200, D))
    a, b = 517, -1290
    mid = O.rope_shift_bf16(kb, a, th)
    two = O.bf16_to_f64(O.rope_shift_bf16(mid, b, th))
    one = O.rope_rotate_f64(O.bf16_to_f64(kb), a + b, th)
    norm = np.sqrt(one[:, : D // 2] ** 2 + one[:, D // 2:] ** 2)
    tol = np.concatenate([norm, norm], axis=1) * 2.0 * 2.0 ** -8 + 1e-30
    assert np.all(np.abs(two - one) <= tol)


def test_p2_identity_delta_zero():
    kb = _rand_bf16((3, 2, 40, 64))
    assert np.array_equal(O.rope_shift_bf16(kb, 0, O.rope_inv_freq(64, 1e4)), kb)


def test_p5_inverse_and_p6_norm():
    D = 128
    th = O.rope_inv_freq(D, 5e5)
    kb = _rand_bf16((300, D))
    delta = 7777
    fwd = O.rope_shift_bf16(kb, delta, th)
    back = O.rope_shift_bf16(fwd, -delta, th)
    k = O.bf16_to_f64(kb)
    norm = np.sqrt(k[:, : D // 2] ** 2 + k[:, D // 2:] ** 2)
    tol = np.concatenate([norm, norm], axis=1) * 2.0 * 2.0 ** -8
    assert np.all(np.abs(O.bf16_to_f64(back) - k) <= tol)
    r = O.rope_rotate_f64(k, delta, th)
    n2 = r[:, : D // 2] ** 2 + r[:, D // 2:] ** 2
    assert np.allclose(n2, norm ** 2, rtol=1e-12, atol=0)
    rb = O.bf16_to_f64(fwd)
    nb = rb[:, : D // 2] ** 2 + rb[:, D // 2:] ** 2
    assert np.all(np.abs(nb - norm ** 2) <= 2.0 ** -6 * norm ** 2 + 1e-30)


def test_p3_one_layer_synthetic_model():
    """north_star pin: for a synthetic one-layer model the re-rotated grafted key equals the fresh
    prefill key W_k x at the new position.  Prefill keys here are computed by the complex form,
    not by the oracle's rotate."""
    D, d_model, n = 64, 96, 37
    th = O.rope_inv_freq(D, 1e4)
    Wk = RNG.standard_normal((D, d_model)) / math.sqrt(d_model)
    x = RNG.standard_normal((n, d_model))
    k_raw = x @ Wk.T

    def prefill_keys(start):
        pos = start + np.arange(n)
        z = (k_raw[:, : D // 2] + 1j * k_raw[:, D // 2:]) * np.exp(1j * pos[:, None] * th[None, :])
        return np.concatenate([z.real, z.imag], axis=1)

    p0, new = 100, 1357
    cached = prefill_keys(p0)                       # what the library would hold (fp64)
    grafted = O.rope_rotate_f64(cached, new - p0, th)
    fresh = prefill_keys(new)
    assert np.max(np.abs(grafted - fresh)) <= 1e-11
    # library copy rounded to bf16 (unit roundoff u = 2^-8): the stored pair is off by <= u*|(a,b)|
    # as a vector, the rotation preserves that, the final rounding adds <= u*|out| <= u*|(a,b)|.
    cached_b = O.f64_to_bf16(cached)
    grafted_b = O.bf16_to_f64(O.rope_shift_bf16(cached_b, new - p0, th))
    norm = np.sqrt(fresh[:, : D // 2] ** 2 + fresh[:, D // 2:] ** 2)
    tol = np.concatenate([norm, norm], axis=1) * 2.0 * 2.0 ** -8
    assert np.all(np.abs(grafted_b - fresh) <= tol)


def test_p7_relative_position_invariance():
    """(R_p q).(R_{s+d} k) = (R_{p-d} q).(R_s k): a grafted key scores like the original at the same distance."""
    D = 64
    th = O.rope_inv_freq(D, 1e4)
    q = RNG.standard_normal((20, D))
    k = RNG.standard_normal((20, D))
    p, s, d = 900, 120, 333
    lhs = np.sum(O.rope_rotate_f64(q, p, th) * O.rope_rotate_f64(O.rope_rotate_f64(k, s, th), d, th), axis=1)
    rhs = np.sum(O.rope_rotate_f64(q, p - d, th) * O.rope_rotate_f64(k, s, th), axis=1)
    assert np.allclose(lhs, rhs, rtol=0, atol=1e-10)


def test_rope_per_row_delta_broadcast():
    D = 16
    th = O.rope_inv_freq(D, 1e4)
    k = RNG.standard_normal((4, D))
    deltas = np.array([0, 5, -9, 1000])
    got = O.rope_rotate_f64(k, deltas, th)
    for r in range(4):
        assert np.array_equal(got[r], O.rope_rotate_f64(k[r], int(deltas[r]), th))


# ----------------------------------------------------------------------------------------------
# attention: brute force, closed forms, library special case
# ----------------------------------------------------------------------------------------------
def _brute_attention(k_bits, v_bits, q_bits, positions, G):
    """pure python loops over scalars; softmax WITHOUT max subtraction (plain definition)."""
    Hkv, cap, D = k_bits.shape
    n, Hq, _ = q_bits.shape
    K = O.bf16_to_f64(k_bits).tolist()
    V = O.bf16_to_f64(v_bits).tolist()
    Q = O.bf16_to_f64(q_bits).tolist()
    out = np.zeros((n, Hq, D))
    for i in range(n):
        for h in range(Hq):
            g = h // G
            ws = []
            for x in range(int(positions[i]) + 1):
                s = 0.0
                for d in range(D):
                    s += Q[i][h][d] * K[g][x][d]
                ws.append(math.exp(s / math.sqrt(D)))
            z = sum(ws)
            for d in range(D):
                acc = 0.0
                for x, w in enumerate(ws):
                    acc += w * V[g][x][d]
                out[i, h, d] = acc / z
    return out


def test_p4_attention_brute_force():
    Hkv, G, D, cap = 2, 2, 8, 23
    kb, vb = _rand_bf16((Hkv, cap, D)), _rand_bf16((Hkv, cap, D))
    qb = _rand_bf16((3, Hkv * G, D))
    pos = np.array([4, 11, 22])
    got = O.patch_attention(kb, vb, qb, pos, G)
    want = _brute_attention(kb, vb, qb, pos, G)
    assert np.allclose(got, want, rtol=1e-12, atol=1e-13)


def test_p9_softmax_closed_forms():
    Hkv, G, D, cap = 2, 3, 16, 50
    kb, vb = _rand_bf16((Hkv, cap, D)), _rand_bf16((Hkv, cap, D))
    V = O.bf16_to_f64(vb)
    pos = np.array([0, 7, 49])
    # q = 0 -> mean of the visible V rows
    q0 = np.zeros((3, Hkv * G, D), np.uint16)
    out = O.patch_attention(kb, vb, q0, pos, G)
    for i, p in enumerate(pos):
        for h in range(Hkv * G):
            assert np.allclose(out[i, h], V[h // G, : p + 1].mean(axis=0), rtol=1e-13, atol=1e-15)
    # one visible token -> exactly that V row
    qb = _rand_bf16((3, Hkv * G, D))
    out = O.patch_attention(kb, vb, qb, pos, G)
    for h in range(Hkv * G):
        assert np.array_equal(out[0, h], V[h // G, 0])
    # convexity: output inside [min, max] of visible V per channel
    for i, p in enumerate(pos):
        for h in range(Hkv * G):
            vis = V[h // G, : p + 1]
            assert np.all(out[i, h] <= vis.max(axis=0) + 1e-12) and np.all(out[i, h] >= vis.min(axis=0) - 1e-12)
    # all V rows equal -> that row
    vconst = np.broadcast_to(vb[:, :1, :], vb.shape).copy()
    out = O.patch_attention(kb, vconst, qb, pos, G)
    for i in range(3):
        for h in range(Hkv * G):
            assert np.allclose(out[i, h], V[h // G, 0], rtol=1e-13, atol=1e-15)
    # a dominant key: q aligned with one key scaled hugely -> output -> that key's V row
    kbig = kb.copy()
    kbig[:, 5, :] = O.f64_to_bf16(np.full((Hkv, D), 64.0))
    qpos = O.f64_to_bf16(np.full((1, Hkv * G, D), 8.0))
    kneg = O.bf16_to_f64(kbig)
    out = O.patch_attention(kbig, vb, qpos, np.array([20]), G)
    # score gap >= 8*64*16/4 - (max other) is enormous; softmax is one-hot to 1e-12
    assert np.all(np.sum(kneg[:, :21], axis=2).argmax(axis=1) == 5)
    for h in range(Hkv * G):
        assert np.allclose(out[0, h], V[h // G, 5], rtol=0, atol=1e-9)


def test_p10_causality():
    Hkv, G, D, cap = 2, 2, 16, 64
    kb, vb = _rand_bf16((Hkv, cap, D)), _rand_bf16((Hkv, cap, D))
    qb = _rand_bf16((2, Hkv * G, D))
    pos = np.array([10, 40])
    a = O.patch_attention(kb, vb, qb, pos, G)
    kb2, vb2 = kb.copy(), vb.copy()
    kb2[:, 41:] = _rand_bf16((Hkv, cap - 41, D))
    vb2[:, 41:] = _rand_bf16((Hkv, cap - 41, D))
    b = O.patch_attention(kb2, vb2, qb, pos, G)
    assert np.array_equal(a, b)
    kb2[:, 11:41] = _rand_bf16((Hkv, 30, D))
    c = O.patch_attention(kb2, vb2, qb, pos, G)
    assert np.array_equal(a[0], c[0]) and not np.array_equal(a[1], c[1])


def test_p12_reduces_to_causal_self_attention_sdpa():
    """empty cache + one patch covering [0, n) = ordinary causal self-attention (torch SDPA, fp64, CPU),
    with GQA expressed the HF way (repeat_interleave of KV heads)."""
    L, Hq, Hkv, D, n = 2, 6, 2, 32, 45
    lib = O.OracleLibrary(L, Hq, Hkv, D, page_size=16, n_pages=64)
    lib.stitch([O.Plan(0, [], [O.Hole(0, n)])])
    qb, kb, vb = _rand_bf16((L, n, Hq, D)), _rand_bf16((L, n, Hkv, D)), _rand_bf16((L, n, Hkv, D))
    out = lib.patch(0, 0, qb, kb, vb, np.arange(n))
    for layer in range(L):
        q = torch.from_numpy(O.bf16_to_f64(qb[layer])).permute(1, 0, 2)[None]
        k = torch.from_numpy(O.bf16_to_f64(kb[layer])).permute(1, 0, 2)[None].repeat_interleave(Hq // Hkv, dim=1)
        v = torch.from_numpy(O.bf16_to_f64(vb[layer])).permute(1, 0, 2)[None].repeat_interleave(Hq // Hkv, dim=1)
        want = torch.nn.functional.scaled_dot_product_attention(q, k, v, is_causal=True)[0].permute(1, 0, 2).numpy()
        assert np.allclose(out[layer], want, rtol=1e-11, atol=1e-12)


# ----------------------------------------------------------------------------------------------
# library state machine: stitch, page tables, scatter, rejection
# ----------------------------------------------------------------------------------------------
def _small_lib(n_pages=256, **kw):
    return O.OracleLibrary(2, 4, 2, 16, page_size=4, n_pages=n_pages, **kw)


def _reg(lib, n, orig_start):
    k, v = _rand_bf16((lib.L, lib.Hkv, n, lib.D)), _rand_bf16((lib.L, lib.Hkv, n, lib.D))
    return lib.segment_register(k, v, orig_start), k, v


def test_stitch_semantics_and_identity():
    lib = _small_lib()
    s0, k0, v0 = _reg(lib, 10, 100)
    s1, k1, v1 = _reg(lib, 7, 0)
    # s0[2:9] -> offset 102 would be delta 0; put it at 5: delta = 5 - 100 - 2 = -97
    lib.stitch([O.Plan(3, [O.PlanEntry(s1, 0, 7, 12), O.PlanEntry(s0, 2, 7, 5)], [O.Hole(0, 5)], 24)])
    t = lib.tasks[3]
    assert t.deltas == [12, -97] and t.capacity == 24 and t.n_tokens == 19
    assert t.page_table == [0, 1, 2, 3, 4, 5]
    assert np.array_equal(t.filled, [False] * 5 + [True] * 14 + [False] * 5)
    assert np.array_equal(t.v[:, :, 12:19], v1) and np.array_equal(t.v[:, :, 5:12], v0[:, :, 2:9])
    assert np.array_equal(t.k[:, :, 5:12], O.rope_shift_bf16(k0[:, :, 2:9], -97, lib.inv_freq))
    # identity graft (P2): one segment at its original position is bit-identical
    lib.stitch([O.Plan(4, [O.PlanEntry(s0, 0, 10, 100)], [], 0)])
    t4 = lib.tasks[4]
    assert t4.deltas == [0]
    assert np.array_equal(t4.k[:, :, 100:110], k0) and np.array_equal(t4.v[:, :, 100:110], v0)
    assert t4.page_table == list(range(6, 6 + 28))          # ceil(110/4) = 28 pages after task 3's six
    # rope_mode 0: pure gather
    lib0 = _small_lib(rope_mode=0)
    s, k, v = _reg(lib0, 9, 50)
    lib0.stitch([O.Plan(0, [O.PlanEntry(s, 0, 9, 3)])])
    assert np.array_equal(lib0.tasks[0].k[:, :, 3:12], k)


def test_page_pool_is_deterministic_lifo():
    pool = O.PagePool(10)
    a = pool.allocate(3)
    b = pool.allocate(4)
    assert a == [0, 1, 2] and b == [3, 4, 5, 6]
    pool.release(a)
    assert pool.allocate(2) == [0, 1]
    pool.release(b)
    assert pool.allocate(5) == [3, 4, 5, 6, 2]
    with pytest.raises(O.OracleError) as e:
        pool.allocate(99)
    assert e.value.status == O.FCG_ERR_OUT_OF_PAGES


def test_p14_plan_rejection_leaves_state_unchanged():
    lib = _small_lib(n_pages=8)
    s0, _, _ = _reg(lib, 10, 0)
    cases = [
        (O.Plan(0, [O.PlanEntry(99, 0, 4, 0)]), O.FCG_ERR_BAD_SEGMENT),
        (O.Plan(0, [O.PlanEntry(s0, 8, 4, 0)]), O.FCG_ERR_RANGE),
        (O.Plan(0, [O.PlanEntry(s0, -1, 4, 0)]), O.FCG_ERR_RANGE),
        (O.Plan(0, [O.PlanEntry(s0, 0, 0, 0)]), O.FCG_ERR_RANGE),
        (O.Plan(0, [O.PlanEntry(s0, 0, 4, -2)]), O.FCG_ERR_RANGE),
        (O.Plan(0, [O.PlanEntry(s0, 0, 4, 0)], [], 3), O.FCG_ERR_RANGE),
        (O.Plan(0, [O.PlanEntry(s0, 0, 4, 0), O.PlanEntry(s0, 4, 4, 3)]), O.FCG_ERR_OVERLAP),
        (O.Plan(0, [O.PlanEntry(s0, 0, 4, 0)], [O.Hole(2, 4)]), O.FCG_ERR_OVERLAP),
        (O.Plan(0, [O.PlanEntry(s0, 0, 4, 0)], [], 1000), O.FCG_ERR_OUT_OF_PAGES),
        (O.Plan(0, [], []), O.FCG_ERR_INVALID_ARG),
        (O.Plan(-1, [O.PlanEntry(s0, 0, 4, 0)]), O.FCG_ERR_BAD_TASK),
    ]
    for plan, status in cases:
        with pytest.raises(O.OracleError) as e:
            lib.stitch([plan])
        assert e.value.status == status, (plan, e.value)
        assert lib.tasks == {} and lib.pool.available() == 8
    # a failing plan in a batch rolls back the whole batch
    good = O.Plan(1, [O.PlanEntry(s0, 0, 4, 0)])
    with pytest.raises(O.OracleError):
        lib.stitch([good, O.Plan(2, [O.PlanEntry(99, 0, 4, 0)])])
    assert lib.tasks == {} and lib.pool.available() == 8
    with pytest.raises(O.OracleError) as e:
        lib.stitch([good, good])
    assert e.value.status == O.FCG_ERR_BAD_TASK
    lib.stitch([good])
    with pytest.raises(O.OracleError) as e:
        lib.stitch([good])
    assert e.value.status == O.FCG_ERR_BAD_TASK
    lib.task_release(1)
    assert lib.pool.available() == 8


def test_patch_scatter_fill_rules_and_sequencing():
    lib = _small_lib()
    s0, _, _ = _reg(lib, 8, 0)
    lib.stitch([O.Plan(0, [O.PlanEntry(s0, 0, 8, 0), O.PlanEntry(s0, 0, 8, 12)], [O.Hole(8, 4), O.Hole(20, 3)])])
    L, Hq, Hkv, D = lib.L, lib.Hq, lib.Hkv, lib.D

    def qkv(n):
        return _rand_bf16((L, n, Hq, D)), _rand_bf16((L, n, Hkv, D)), _rand_bf16((L, n, Hkv, D))

    q, k, v = qkv(3)
    # attending over the unfilled mid hole is an error and changes nothing
    before = lib.tasks[0].k.copy()
    with pytest.raises(O.OracleError) as e:
        lib.patch(0, 0, q, k, v, [20, 21, 22])
    assert e.value.status == O.FCG_ERR_UNFILLED and np.array_equal(before, lib.tasks[0].k)
    # positions beyond the capacity (23) append (R25, pinned in test_oracle_pins_r2.py) -- here the hole at 20
    # is still unfilled, so the call fails as UNFILLED; RANGE is left for negative positions
    for bad, status in (([9, 8, 10], O.FCG_ERR_INVALID_ARG), ([8, 8, 9], O.FCG_ERR_INVALID_ARG),
                        ([21, 22, 23], O.FCG_ERR_UNFILLED), ([-1, 0, 1], O.FCG_ERR_RANGE)):
        with pytest.raises(O.OracleError) as e:
            lib.patch(0, 0, q, k, v, bad)
        assert e.value.status == status
    with pytest.raises(O.OracleError) as e:
        lib.patch(7, 0, q, k, v, [8, 9, 10])
    assert e.value.status == O.FCG_ERR_BAD_TASK
    # a partial fill of the mid hole is fine as long as every query only sees filled positions
    q2, k2, v2 = qkv(2)
    lib.patch(0, 0, q2, k2, v2, [8, 9])
    with pytest.raises(O.OracleError) as e:
        lib.patch(0, 0, q2, k2, v2, [11, 20])          # 10 still unfilled
    assert e.value.status == O.FCG_ERR_UNFILLED
    q4, k4, v4 = qkv(5)
    out = lib.patch(0, 0, q4, k4, v4, [10, 11, 20, 21, 22])
    t = lib.tasks[0]
    assert t.filled.all() and t.n_tokens == 23
    for layer in range(L):
        assert np.array_equal(t.k[layer][:, [10, 11, 20, 21, 22]], np.transpose(k4[layer], (1, 0, 2)))
        assert np.array_equal(t.v[layer][:, [8, 9]], np.transpose(v2[layer], (1, 0, 2)))
        # scatter happens-before attention, later tokens see earlier ones of the same call
        want = O.patch_attention(t.k[layer], t.v[layer], q4[layer], [10, 11, 20, 21, 22], lib.G)
        assert np.array_equal(out[layer], want)
    # layer sub-range call only touches those layers
    q1, k1, v1 = _rand_bf16((1, 1, Hq, D)), _rand_bf16((1, 1, Hkv, D)), _rand_bf16((1, 1, Hkv, D))
    k_l0 = t.k[0].copy()
    lib.patch(0, 1, q1, k1, v1, [22])
    assert np.array_equal(t.k[0], k_l0) and np.array_equal(t.k[1][:, 22], k1[0, 0])


def test_p11_page_size_does_not_change_logical_results():
    """page size only changes the page table, never the stitched bytes or the attention output."""
    outs = []
    for P in (2, 4, 16):
        lib = O.OracleLibrary(1, 4, 2, 16, page_size=P, n_pages=512)
        rs = np.random.default_rng(5)
        k = rs.integers(0x3C00, 0x4080, (1, 2, 30, 16)).astype(np.uint16)
        v = rs.integers(0x3C00, 0x4080, (1, 2, 30, 16)).astype(np.uint16)
        s = lib.segment_register(k, v, 11)
        lib.stitch([O.Plan(0, [O.PlanEntry(s, 3, 20, 0)], [O.Hole(20, 2)])])
        q = rs.integers(0x3C00, 0x4080, (1, 2, 4, 16)).astype(np.uint16)
        kk = rs.integers(0x3C00, 0x4080, (1, 2, 2, 16)).astype(np.uint16)
        out = lib.patch(0, 0, q, kk, kk, [20, 21])
        outs.append((lib.tasks[0].k.copy(), lib.tasks[0].v.copy(), out))
        assert len(lib.tasks[0].page_table) == -(-22 // P)
    for o in outs[1:]:
        assert all(np.array_equal(a, b) for a, b in zip(outs[0], o))


# ----------------------------------------------------------------------------------------------
# NEXT rows: interleaved pairs, suffix re-graft (task_shift), segment extraction
# ----------------------------------------------------------------------------------------------
def _complex_shift_bits(k_bits, delta, th, interleaved=False):
    """independent restatement of a key shift: complex multiplication in numpy complex128, one RNE."""
    x = O.bf16_to_f64(k_bits)
    half = x.shape[-1] // 2
    z = (x[..., 0::2] + 1j * x[..., 1::2]) if interleaved else (x[..., :half] + 1j * x[..., half:])
    z = z * np.exp(1j * delta * th)
    out = np.empty_like(x)
    if interleaved:
        out[..., 0::2], out[..., 1::2] = z.real, z.imag
    else:
        out[..., :half], out[..., half:] = z.real, z.imag
    return O.f64_to_bf16(out)


def _pair_err_ok(a_bits, b_bits, c):
    """|a - b| <= c * 2^-9 * |pair| per component (half-split pairs): the error of a rounded rotation is bounded
    relative to the norm of its rotation pair, not to the component itself (a small component next to a large one
    moves by many of its own ulps).  Two roundings with a rotation in between: c = 1 + sqrt(2) < 3."""
    a, b = O.bf16_to_f64(a_bits), O.bf16_to_f64(b_bits)
    half = a.shape[-1] // 2
    norm = np.sqrt(b[..., :half] ** 2 + b[..., half:] ** 2)
    tol = np.concatenate([norm, norm], axis=-1) * c * 2.0 ** -9
    return bool(np.all(np.abs(a - b) <= tol))


def test_rope_interleaved_matches_complex_multiplication_and_permuted_half_split():
    D = 16
    th = O.rope_inv_freq(D, 5e5)
    k = RNG.standard_normal((6, D))
    perm = np.concatenate([np.arange(0, D, 2), np.arange(1, D, 2)])       # interleaved -> half-split order
    for delta in (-1234, -1, 0, 1, 513, 32767):
        got = O.rope_rotate_f64(k, delta, th, O.ROPE_INTERLEAVED)
        for r in range(6):
            for j in range(D // 2):
                z = complex(k[r, 2 * j], k[r, 2 * j + 1]) * cmath.exp(1j * delta * th[j])
                assert math.isclose(got[r, 2 * j], z.real, rel_tol=0, abs_tol=1e-12)
                assert math.isclose(got[r, 2 * j + 1], z.imag, rel_tol=0, abs_tol=1e-12)
        # the two layouts are the same rotation up to the fixed permutation of the head dimension
        via_half = O.rope_rotate_f64(k[:, perm], delta, th, O.ROPE_HALF_SPLIT)
        assert np.array_equal(got[:, perm], via_half)
    # D = 2 has a single pair: both layouts coincide with the closed form (cos d, sin d) of (1, 0)
    one = O.rope_rotate_f64(np.array([[1.0, 0.0]]), 3, np.array([1.0]), O.ROPE_INTERLEAVED)
    assert np.allclose(one, [[math.cos(3), math.sin(3)]], rtol=0, atol=1e-15)
    with pytest.raises(O.OracleError):
        O.rope_rotate_f64(k, 1, th, 0)


def test_interleaved_library_stitch():
    lib = _small_lib(rope_mode=O.ROPE_INTERLEAVED)
    s, k, v = _reg(lib, 9, 40)
    lib.stitch([O.Plan(0, [O.PlanEntry(s, 1, 8, 3)])])
    t = lib.tasks[0]
    assert t.deltas == [3 - 40 - 1]
    assert np.array_equal(t.k[:, :, 3:11], _complex_shift_bits(k[:, :, 1:9], -38, lib.inv_freq, interleaved=True))
    assert np.array_equal(t.v[:, :, 3:11], v[:, :, 1:9])


def test_task_shift_semantics_pages_and_rejection():
    """Hand-computed paging example (P = 4, pool of 8): capacity 12 -> pages [0,1,2]; moving [4,8) to [6,10)
    re-pages logical pages 1 and 2 onto fresh pages 3 and 4, and returns 1, 2 to the pool in that order.
    (max_task_tokens = 12 here: a destination beyond the capacity would otherwise append, R25.)"""
    lib = _small_lib(n_pages=8, max_task_tokens=12)
    s, k, v = _reg(lib, 8, 0)
    lib.stitch([O.Plan(0, [O.PlanEntry(s, 0, 8, 0)], [], 12)])
    t = lib.tasks[0]
    assert t.page_table == [0, 1, 2] and t.n_tokens == 8
    k_before, v_before = t.k.copy(), t.v.copy()
    lib.task_shift(0, 4, 4, 6)
    assert t.page_table == [0, 3, 4]
    assert lib.pool.allocate(2) == [1, 2]
    assert np.array_equal(t.filled, [True] * 4 + [False] * 2 + [True] * 4 + [False] * 2)
    assert t.n_tokens == 10
    # V is a bit copy, K is the delta rotation of the bits that were in the cache (independent complex form)
    assert np.array_equal(t.v[:, :, 6:10], v_before[:, :, 4:8])
    assert np.array_equal(t.k[:, :, 6:10], _complex_shift_bits(k_before[:, :, 4:8], 2, lib.inv_freq))
    # everything outside the destination range is untouched (incl. the vacated source slots' stale bits)
    keep = np.r_[0:6, 10:12]
    assert np.array_equal(t.k[:, :, keep], k_before[:, :, keep]) and np.array_equal(t.v[:, :, keep], v_before[:, :, keep])
    # rejections change nothing
    snap = (list(t.page_table), t.filled.copy(), t.k.copy(), lib.pool.available())
    for args, status in (((0, 4, 2, 6), O.FCG_ERR_UNFILLED),        # source [4,6) is a hole now
                         ((0, 6, 4, 9), O.FCG_ERR_RANGE),           # 9 + 4 > max_task_tokens 12
                         ((0, -1, 2, 0), O.FCG_ERR_RANGE),
                         ((0, 0, 0, 2), O.FCG_ERR_RANGE),
                         ((7, 0, 2, 2), O.FCG_ERR_BAD_TASK)):
        with pytest.raises(O.OracleError) as e:
            lib.task_shift(*args)
        assert e.value.status == status
    lib.pool.allocate(lib.pool.available())                          # drain the pool
    with pytest.raises(O.OracleError) as e:
        lib.task_shift(0, 0, 4, 1)
    assert e.value.status == O.FCG_ERR_OUT_OF_PAGES
    assert snap[0] == t.page_table and np.array_equal(snap[1], t.filled) and np.array_equal(snap[2], t.k)
    # delta 0 is a no-op even with an empty pool
    lib.task_shift(0, 0, 4, 0)
    assert snap[0] == t.page_table and np.array_equal(snap[1], t.filled)


def test_task_shift_overlapping_moves_and_round_trip():
    lib = _small_lib()
    s, k, v = _reg(lib, 40, 17)
    lib.stitch([O.Plan(0, [O.PlanEntry(s, 0, 40, 5)], [O.Hole(0, 5)], 64)])
    t = lib.tasks[0]
    k0, v0 = t.k[:, :, 5:45].copy(), t.v[:, :, 5:45].copy()
    lib.task_shift(0, 20, 25, 23)            # overlapping move to the right (longer x_mid): +3
    assert np.array_equal(t.v[:, :, 23:48], v0[:, :, 15:40])
    assert np.array_equal(t.k[:, :, 23:48], _complex_shift_bits(k0[:, :, 15:40], 3, lib.inv_freq))
    assert not t.filled[20:23].any() and t.filled[23:48].all() and t.filled[5:20].all()
    lib.task_shift(0, 23, 25, 20)            # and back (shorter x_mid): -3
    assert np.array_equal(t.v[:, :, 5:45], v0)
    assert _pair_err_ok(t.k[:, :, 5:45], k0, 3.0)             # two roundings, one per move
    assert np.array_equal(t.k[:, :, 5:20], k0[:, :, :15])     # the untouched prefix is bit-identical
    assert t.filled[5:45].all() and not t.filled[45:].any()


def test_task_shift_equals_fresh_prefill_for_synthetic_model():
    """north_star's synthetic one-layer model, for the re-grafted suffix: keys moved by task_shift equal the
    keys a prefill at the new positions would produce, up to the stored-bf16 and output roundings."""
    D, d_model, n = 16, 24, 12
    lib = O.OracleLibrary(1, 1, 1, D, page_size=4, n_pages=64)
    th = lib.inv_freq
    Wk = RNG.standard_normal((D, d_model)) / math.sqrt(d_model)
    x = RNG.standard_normal((n, d_model))
    k_raw = x @ Wk.T

    def prefill(start):
        pos = start + np.arange(n)
        z = (k_raw[:, : D // 2] + 1j * k_raw[:, D // 2:]) * np.exp(1j * pos[:, None] * th[None, :])
        return np.concatenate([z.real, z.imag], axis=1)

    sid = lib.segment_register(O.f64_to_bf16(prefill(30))[None, None], _rand_bf16((1, 1, n, D)), 30)
    lib.stitch([O.Plan(0, [O.PlanEntry(sid, 0, n, 30)], [O.Hole(0, 30)], 64)])      # identity graft at 30
    lib.task_shift(0, 36, 6, 41)                                                   # suffix [36,42) -> [41,47)
    got = O.bf16_to_f64(lib.tasks[0].k[0, 0, 41:47])
    fresh = prefill(35)[6:]                                                        # tokens 6.. at positions 41..
    norm = np.sqrt(fresh[:, : D // 2] ** 2 + fresh[:, D // 2:] ** 2)
    tol = np.concatenate([norm, norm], axis=1) * 2.0 * 2.0 ** -8
    assert np.all(np.abs(got - fresh) <= tol)


def test_segment_extract_round_trips():
    lib = _small_lib()
    s, k, v = _reg(lib, 30, 100)
    lib.stitch([O.Plan(0, [O.PlanEntry(s, 0, 30, 7)], [O.Hole(0, 7)], 40)])
    t = lib.tasks[0]
    # (a) keep the encoding of the cache: bit copy, and stitching it back at the same place is the identity
    e0 = lib.segment_extract(0, 12, 10, 12)
    assert e0 == 1 and lib.segments[e0].orig_start == 12 and lib.segments[e0].n_tokens == 10
    assert np.array_equal(lib.segments[e0].k, t.k[:, :, 12:22]) and np.array_equal(lib.segments[e0].v, t.v[:, :, 12:22])
    lib.stitch([O.Plan(1, [O.PlanEntry(e0, 0, 10, 12)], [O.Hole(0, 12)], 24)])
    assert lib.tasks[1].deltas == [0]
    assert np.array_equal(lib.tasks[1].k[:, :, 12:22], t.k[:, :, 12:22])
    # (b) canonical form: un-rotated to position 0 (independent complex form), V untouched
    e1 = lib.segment_extract(0, 12, 10, 0)
    assert lib.segments[e1].orig_start == 0
    assert np.array_equal(lib.segments[e1].k, _complex_shift_bits(t.k[:, :, 12:22], -12, lib.inv_freq))
    assert np.array_equal(lib.segments[e1].v, t.v[:, :, 12:22])
    # grafting the canonical segment back where it came from returns the keys up to two roundings
    lib.stitch([O.Plan(2, [O.PlanEntry(e1, 0, 10, 12)], [O.Hole(0, 12)], 24)])
    assert lib.tasks[2].deltas == [12]
    assert _pair_err_ok(lib.tasks[2].k[:, :, 12:22], t.k[:, :, 12:22], 3.0)
    # rejections
    for args, status in (((0, 0, 10, 0), O.FCG_ERR_UNFILLED), ((0, 35, 10, 0), O.FCG_ERR_RANGE),
                         ((0, 12, 10, -1), O.FCG_ERR_INVALID_ARG), ((9, 12, 10, 0), O.FCG_ERR_BAD_TASK)):
        n_seg = len(lib.segments)
        with pytest.raises(O.OracleError) as e:
            lib.segment_extract(*args)
        assert e.value.status == status and len(lib.segments) == n_seg


def test_segment_residency_state_machine():
    """NEXT-3: residency is bookkeeping only -- the same plan over resident and offloaded segments gives the same
    cache bits; offload / prefetch are idempotent; ids of offloaded segments stay taken until released."""
    lib = _small_lib()
    s0, k0, v0 = _reg(lib, 12, 5)
    s1, k1, v1 = _reg(lib, 9, 0)
    plan = lambda tid: O.Plan(tid, [O.PlanEntry(s0, 1, 10, 0), O.PlanEntry(s1, 0, 9, 10)])
    lib.stitch([plan(0)])
    assert lib.segment_info(s0) == (12, 5, True)
    lib.segment_offload(s0), lib.segment_offload(s0)
    assert lib.segment_info(s0) == (12, 5, False) and lib.segment_info(s1)[2] is True
    lib.stitch([plan(1)])
    assert np.array_equal(lib.tasks[0].k, lib.tasks[1].k) and np.array_equal(lib.tasks[0].v, lib.tasks[1].v)
    assert _reg(lib, 3, 0)[0] == 2                       # the offloaded segment still owns id 0
    lib.segment_prefetch(s0), lib.segment_prefetch(s0)
    assert lib.segment_info(s0) == (12, 5, True)
    lib.segment_offload(s1)
    lib.segment_release(s1)
    assert _reg(lib, 3, 0)[0] == s1
    for fn in (lib.segment_offload, lib.segment_prefetch, lib.segment_info):
        with pytest.raises(O.OracleError) as e:
            fn(77)
        assert e.value.status == O.FCG_ERR_BAD_SEGMENT


def test_patch_rope_is_rotation_to_absolute_positions_then_patch():
    """patch_rope == rotate q_i, k_i to p_i (independent complex form, one rounding) then patch; and what it computes
    depends on relative positions only (P7 through the whole call): the same tokens patched at positions c.. instead
    of 0.. give the same output once the mass of the c zero-key / zero-value filler tokens is accounted for."""
    lib = _small_lib()
    L, Hq, Hkv, D = lib.L, lib.Hq, lib.Hkv, lib.D
    n = 9
    q, k, v = _rand_bf16((L, n, Hq, D)), _rand_bf16((L, n, Hkv, D)), _rand_bf16((L, n, Hkv, D))
    pos = np.arange(n)
    lib.stitch([O.Plan(0, [], [O.Hole(0, n)], n)])
    out = lib.patch_rope(0, 0, q, k, v, pos)
    manual_q = np.stack([_complex_shift_bits(q[:, i], int(p), lib.inv_freq) for i, p in enumerate(pos)], axis=1)
    manual_k = np.stack([_complex_shift_bits(k[:, i], int(p), lib.inv_freq) for i, p in enumerate(pos)], axis=1)
    assert np.array_equal(np.transpose(lib.tasks[0].k[:, :, pos], (0, 2, 1, 3)), manual_k)
    lib2 = _small_lib()
    lib2.stitch([O.Plan(0, [], [O.Hole(0, n)], n)])
    assert np.array_equal(lib2.patch(0, 0, manual_q, manual_k, v, pos), out)
    # shifted by c = 40 behind filler tokens with zero keys (score 0) and zero values
    lib3 = _small_lib()
    c = 40
    lib3.stitch([O.Plan(0, [], [O.Hole(0, c + n)], c + n)])
    zeros = lambda h: np.zeros((L, c, h, D), np.uint16)
    lib3.patch(0, 0, zeros(Hq), zeros(Hkv), zeros(Hkv), np.arange(c))
    out_shift = lib3.patch_rope(0, 0, q, k, v, np.arange(c, c + n))
    qf, kf = O.bf16_to_f64(q), O.bf16_to_f64(k)
    for li in range(L):
        for i in range(n):
            for h in range(Hq):
                g = h // lib.G
                s_rel = np.array([np.dot(O.rope_rotate_f64(qf[li, i, h], i, lib.inv_freq), O.rope_rotate_f64(kf[li, x, g], x, lib.inv_freq))
                                  for x in range(i + 1)]) / math.sqrt(D)
                m = max(s_rel.max(), 0.0)
                w = np.exp(s_rel - m)
                ref = (w @ O.bf16_to_f64(v[li, : i + 1, g])) / (w.sum() + c * math.exp(-m))
                assert np.allclose(out_shift[li, i, h], ref, rtol=0, atol=0.06), (li, i, h)
    # rope_mode NONE: patch_rope is patch
    lib0 = _small_lib(rope_mode=0)
    lib0.stitch([O.Plan(0, [], [O.Hole(0, n)], n)])
    a = lib0.patch_rope(0, 0, q, k, v, np.arange(n))
    lib0.task_release(0)
    lib0.stitch([O.Plan(0, [], [O.Hole(0, n)], n)])
    assert np.array_equal(a, lib0.patch(0, 0, q, k, v, np.arange(n)))


def test_boundary_positions_by_hand():
    """entries at 0 (n 10), 14 (n 7), 21 (n 2) and a hole [10, 14): width 3 -> the first 3 tokens of the entries that
    do not start at 0, the short one contributing only its 2."""
    lib = _small_lib()
    s0, _, _ = _reg(lib, 10, 0)
    s1, _, _ = _reg(lib, 7, 50)
    lib.stitch([O.Plan(0, [O.PlanEntry(s0, 0, 10, 0), O.PlanEntry(s1, 0, 7, 14), O.PlanEntry(s0, 3, 2, 21)], [O.Hole(10, 4)], 30)])
    assert lib.task_boundary_positions(0, 3) == [14, 15, 16, 21, 22]
    assert lib.task_boundary_positions(0, 1) == [14, 21]
    assert lib.task_boundary_positions(0, 100) == list(range(14, 23))
    with pytest.raises(O.OracleError):
        lib.task_boundary_positions(0, 0)
    with pytest.raises(O.OracleError):
        lib.task_boundary_positions(5, 2)
