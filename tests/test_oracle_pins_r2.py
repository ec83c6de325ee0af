"""Pins of the oracle functions added in round 2 (no GPU, no libfcg.so compute calls):

* appends beyond the reserved capacity take pages on demand (R25): hand-computed
  page tables (tests/golden/page_growth.txt) and the equivalence "growing == having reserved the room up front";
* fp8 (e4m3) segment storage (R26): the codec against hand-worked values
  (tests/golden/fp8_e4m3.txt), against torch's float8_e4m3fn type (a library routine), and against brute force
  over the 256-code table; the row scale by hand; stitching from fp8 storage against the already pinned bf16
  stitch of the de-quantised segment.
"""
import os

import numpy as np
import pytest
import torch

from oracle import fcg_oracle as O

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _rand_bf16(shape, seed=0, scale=1.0):
    rs = np.random.default_rng(seed)
    return O.f64_to_bf16(rs.standard_normal(shape) * scale)


def growth_script():
    """(op, args, status, table, capacity, free) rows of tests/golden/page_growth.txt"""
    rows = []
    with open(os.path.join(GOLDEN, "page_growth.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            op, status, table, cap, free = [x.strip() for x in line.split(";")]
            op = op.split()
            rows.append((op[0], [int(x) for x in op[1:]], int(status), [int(x) for x in table.split()], int(cap), int(free)))
    return rows


# ------------------------------------------------------------------------------------------------
# R25: on-demand growth
# ------------------------------------------------------------------------------------------------
def test_growth_page_tables_by_hand():
    L, Hq, Hkv, D = 1, 2, 1, 8
    lib = O.OracleLibrary(L, Hq, Hkv, D, page_size=4, n_pages=8, max_task_tokens=16)
    sid = lib.segment_register(_rand_bf16((L, Hkv, 6, D), 1), _rand_bf16((L, Hkv, 6, D), 2), 0)
    for op, args, status, table, cap, free in growth_script():
        got = O.FCG_OK
        try:
            if op == "stitch":
                t, c = args
                lib.stitch([O.Plan(t, [O.PlanEntry(sid, 0, min(c, 6), 0)], [O.Hole(6, c - 6)] if c > 6 else [], c)])
            elif op == "release":
                lib.task_release(args[0])
            elif op == "patch":
                t, pos = args[0], args[1:]
                n = len(pos)
                lib.patch(t, 0, _rand_bf16((L, n, Hq, D), 3), _rand_bf16((L, n, Hkv, D), 4), _rand_bf16((L, n, Hkv, D), 5), pos)
        except O.OracleError as e:
            got = e.status
        what = f"{op} {args}"
        assert got == status, what
        assert lib.tasks[0].page_table == table and lib.tasks[0].capacity == cap, what
        assert lib.pool.available() == free, what
        assert lib.tasks[0].k.shape[2] == cap == lib.tasks[0].filled.size


def test_growing_equals_reserving_up_front():
    """A task that grows token by token holds the same logical cache and gives the same attention outputs as a
    task whose plan reserved the room from the start (capacity_tokens): growth changes paging, not values."""
    L, Hq, Hkv, D, P = 2, 4, 2, 16, 4
    k, v = _rand_bf16((L, Hkv, 10, D), 1), _rand_bf16((L, Hkv, 10, D), 2)
    grow = O.OracleLibrary(L, Hq, Hkv, D, page_size=P, n_pages=64)
    resv = O.OracleLibrary(L, Hq, Hkv, D, page_size=P, n_pages=64)
    for lib, cap in ((grow, 0), (resv, 23)):
        s = lib.segment_register(k, v, 7)
        lib.stitch([O.Plan(0, [O.PlanEntry(s, 0, 10, 0)], [], cap)])
    assert grow.tasks[0].capacity == 10 and len(grow.tasks[0].page_table) == 3
    steps = [[10], [11, 12], [13], [14, 15, 16, 17, 18], [19], [20, 21, 22]]
    for i, pos in enumerate(steps):
        n = len(pos)
        q, kk, vv = _rand_bf16((L, n, Hq, D), 10 + i), _rand_bf16((L, n, Hkv, D), 20 + i), _rand_bf16((L, n, Hkv, D), 30 + i)
        a = grow.patch(0, 0, q, kk, vv, pos)
        b = resv.patch(0, 0, q, kk, vv, pos)
        assert np.array_equal(a, b)
        tg = grow.tasks[0]
        assert tg.capacity == pos[-1] + 1 and tg.n_tokens == pos[-1] + 1
        assert len(tg.page_table) == -(-tg.capacity // P) and tg.page_table == list(range(len(tg.page_table)))
    tg, tr = grow.tasks[0], resv.tasks[0]
    assert np.array_equal(tg.k, tr.k) and np.array_equal(tg.v, tr.v) and np.array_equal(tg.filled, tr.filled)
    assert tg.page_table == tr.page_table            # one live task: both end up with pages 0..5
    # a gap is not an append: 24 would leave 23 unfilled
    q, kk, vv = _rand_bf16((L, 1, Hq, D), 1), _rand_bf16((L, 1, Hkv, D), 2), _rand_bf16((L, 1, Hkv, D), 3)
    with pytest.raises(O.OracleError) as e:
        grow.patch(0, 0, q, kk, vv, [24])
    assert e.value.status == O.FCG_ERR_UNFILLED and grow.tasks[0].capacity == 23


def test_task_shift_beyond_capacity_grows_by_hand():
    """P = 4, pool of 16, one task of capacity 10 -> pages [0, 1, 2], next free pages 3, 4, 5, ...
    shift [4, 8) -> [17, 21): destination logical pages 4, 5; logical page 3 is a gap page.  New physical pages in
    ascending logical order: lp3 -> 3, lp4 -> 4, lp5 -> 5; nothing existed there, nothing is released.
    then shift [0, 4) -> [9, 13): destination logical pages 2 (exists, physical 2) and 3 (exists, physical 3):
    lp2 -> 6, lp3 -> 7; pages 2 and 3 go back (re-issued in that order)."""
    L, Hq, Hkv, D = 1, 2, 1, 8
    lib = O.OracleLibrary(L, Hq, Hkv, D, page_size=4, n_pages=16, max_task_tokens=24)
    k, v = _rand_bf16((L, Hkv, 10, D), 1), _rand_bf16((L, Hkv, 10, D), 2)
    s = lib.segment_register(k, v, 0)
    lib.stitch([O.Plan(0, [O.PlanEntry(s, 0, 10, 0)])])
    t = lib.tasks[0]
    before_k, before_v = t.k.copy(), t.v.copy()
    lib.task_shift(0, 4, 4, 17)
    t = lib.tasks[0]
    assert t.page_table == [0, 1, 2, 3, 4, 5] and t.capacity == 21 and t.n_tokens == 21 and lib.pool.available() == 10
    assert np.array_equal(t.filled, [True] * 4 + [False] * 4 + [True] * 2 + [False] * 7 + [True] * 4)
    assert np.array_equal(t.v[:, :, 17:21], before_v[:, :, 4:8])
    assert np.array_equal(t.k[:, :, 17:21], O.rope_shift_bf16(before_k[:, :, 4:8], 13, lib.inv_freq))
    lib.task_shift(0, 0, 4, 9)
    assert t.page_table == [0, 1, 6, 7, 4, 5] and t.capacity == 21 and lib.pool.available() == 10
    assert lib.pool.allocate(2) == [2, 3]
    # destination beyond max_task_tokens: RANGE, nothing changes
    with pytest.raises(O.OracleError) as e:
        lib.task_shift(0, 8, 2, 23)
    assert e.value.status == O.FCG_ERR_RANGE and t.page_table == [0, 1, 6, 7, 4, 5]


def test_growth_then_release_returns_every_page():
    lib = O.OracleLibrary(1, 2, 1, 8, page_size=4, n_pages=8)
    s = lib.segment_register(_rand_bf16((1, 1, 4, 8), 1), _rand_bf16((1, 1, 4, 8), 2), 0)
    lib.stitch([O.Plan(0, [O.PlanEntry(s, 0, 4, 0)])])
    for p in range(4, 14):
        lib.patch(0, 0, _rand_bf16((1, 1, 2, 8), p), _rand_bf16((1, 1, 1, 8), p), _rand_bf16((1, 1, 1, 8), p), [p])
    assert lib.tasks[0].page_table == [0, 1, 2, 3] and lib.pool.available() == 4
    lib.task_release(0)
    assert lib.pool.available() == 8 and lib.pool.allocate(8) == list(range(8))


# ------------------------------------------------------------------------------------------------
# R26: fp8 e4m3 storage
# ------------------------------------------------------------------------------------------------
def fp8_golden():
    code, rnd, rows = [], [], []
    with open(os.path.join(GOLDEN, "fp8_e4m3.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            kind, rest = line.split(None, 1)
            if kind == "code":
                c, v = rest.split()
                code.append((int(c, 16), float(v)))
            elif kind == "round":
                v, c = rest.split()
                rnd.append((float(v), int(c, 16)))
            elif kind == "row":
                bits, e, codes, vals = [x.split() for x in rest.split(";")]
                rows.append(([int(b, 16) for b in bits], int(e[0]), [int(c, 16) for c in codes], [float(x) for x in vals]))
    return code, rnd, rows


def test_e4m3_golden_values_rounding_and_rows():
    code, rnd, rows = fp8_golden()
    assert len(code) >= 20 and len(rnd) >= 12 and len(rows) >= 3
    for c, v in code:
        got = O.e4m3_to_f64(np.asarray([c], np.uint8))[0]
        assert (np.isnan(got) and np.isnan(v)) or (got == v and np.signbit(got) == np.signbit(v)), hex(c)
    for v, c in rnd:
        assert O.f64_to_e4m3(np.asarray([v]))[0] == c, v
    for bits, e, codes, vals in rows:
        b = np.asarray(bits, np.uint16)
        got_codes, got_e = O.fp8_quantize_rows(b[None, :])
        assert got_e[0] == e and got_codes[0].tolist() == codes, bits
        assert O.fp8_dequantize_rows(got_codes, got_e)[0].tolist() == vals


def test_e4m3_decode_matches_torch_float8_for_all_256_codes():
    c = np.arange(256, dtype=np.uint8)
    mine = O.e4m3_to_f64(c)
    lib = torch.from_numpy(c.copy()).view(torch.float8_e4m3fn).to(torch.float64).numpy()
    assert np.array_equal(np.isnan(mine), np.isnan(lib)) and np.isnan(mine).sum() == 2
    ok = ~np.isnan(mine)
    assert np.array_equal(mine[ok], lib[ok]) and np.array_equal(np.signbit(mine[ok]), np.signbit(lib[ok]))
    # every finite code is a fixed point of the encoder; the grid is symmetric and strictly increasing in the code
    assert np.array_equal(O.f64_to_e4m3(mine[ok]), c[ok])
    pos = mine[:0x7F]
    assert np.all(np.diff(pos) > 0) and pos[-1] == 448.0 and np.array_equal(mine[0x80:0xFF], -pos)


def test_e4m3_encode_is_nearest_even_by_brute_force_and_matches_torch_in_range():
    grid = O.e4m3_to_f64(np.arange(0x7F, dtype=np.uint8))            # the 127 non-negative finite values, ascending
    rs = np.random.default_rng(7)
    x = np.concatenate([rs.standard_normal(20000) * s for s in (1e-3, 0.05, 1.0, 30.0, 200.0)])
    mids = (grid[1:] + grid[:-1]) / 2                                  # every tie of the format
    x = np.concatenate([x, mids, -mids, np.nextafter(mids, 0), np.nextafter(mids, 1e9), grid, [0.0, -0.0, 500.0, -1e30]])
    got = O.f64_to_e4m3(x)
    a = np.minimum(np.abs(x), 448.0)                                   # satfinite
    d = np.abs(a[:, None] - grid[None, :])
    best = d.min(axis=1)
    cand = d == best[:, None]
    # nearest; on a tie (two candidates) the one with the even code (mantissa LSB 0)
    want = np.where(cand.sum(axis=1) == 1, cand.argmax(axis=1),
                    np.where(cand.argmax(axis=1) % 2 == 0, cand.argmax(axis=1), cand.argmax(axis=1) + 1))
    assert np.array_equal(got & 0x7F, want.astype(np.uint8))
    assert np.array_equal((got & 0x80) != 0, np.signbit(x))
    # torch's conversion (fp32 -> float8_e4m3fn, RNE) is an independent witness wherever no saturation is involved
    inr = np.abs(x) <= 448.0
    x32 = x[inr].astype(np.float32)                                    # the witness sees the fp32 value
    lib = torch.from_numpy(x32).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    assert np.array_equal(O.f64_to_e4m3(x32.astype(np.float64)), lib)


def test_fp8_row_exponent_and_error_bounds():
    # e is the smallest integer with amax <= 448 * 2^e: check the definition itself, exhaustively over bf16 amax
    bits = np.arange(0x0001, 0x7F80, dtype=np.uint16)                  # every positive finite bf16
    x = O.bf16_to_f64(bits)
    e = O.fp8_row_exponent(x[:, None])
    un = (e > -127) & (e < 127)
    assert np.all(x[un] <= 448.0 * np.ldexp(1.0, e[un])) and np.all(x[un] > 448.0 * np.ldexp(1.0, e[un] - 1))
    assert np.all(x[e == -127] <= 448.0 * 2.0 ** -127) and e.min() == -127 and e.max() <= 127
    assert O.fp8_row_exponent(np.zeros((3, 8)))[0] == 0
    assert O.fp8_row_exponent(np.asarray([[1.0, np.inf, np.nan, -2.0]]))[0] == O.fp8_row_exponent(np.asarray([[2.0]]))[0]
    # quantisation error of N(0,1) rows: <= 2^-4 relative for elements that land in the normal range,
    # <= 2^-10 * 2^e absolute below it; the row maximum keeps at least 3 mantissa bits
    k = _rand_bf16((64, 128), 3)
    codes, ex = O.fp8_quantize_rows(k)
    dq = O.fp8_dequantize_rows(codes, ex)
    xf = O.bf16_to_f64(k)
    err = np.abs(dq - xf)
    scale = np.ldexp(1.0, ex)[:, None]
    assert np.all(err <= np.maximum(np.abs(xf) * 2.0 ** -4, scale * 2.0 ** -10))
    assert np.all(np.abs(dq).max(axis=1) > 224.0 * scale[:, 0] * (1 - 2.0 ** -4))
    # non-finite elements become NaN, the others are quantised as if they were not there
    k2 = k.copy()
    k2[0, 5], k2[0, 9] = 0x7F80, 0x7FC0
    c2, e2 = O.fp8_quantize_rows(k2)
    keep = np.ones(128, bool)
    keep[[5, 9]] = False
    assert e2[0] == ex[0] and c2[0, 5] == 0x7F and c2[0, 9] == 0x7F and np.array_equal(c2[0, keep], codes[0, keep])


@pytest.mark.parametrize("rope_mode", [1, 2, 0])
def test_fp8_stitch_equals_bf16_stitch_of_the_dequantised_segment(rope_mode):
    """code * 2^e has <= 4 significant bits, so (outside the deepest subnormals) it IS a bf16 value: a library that
    holds the de-quantised segment in bf16 must stitch to the same bits -- which ties the fp8 path to the pinned
    bf16 path (closed forms, complex multiplication, group law ...)."""
    L, Hq, Hkv, D, P = 2, 4, 2, 32, 4
    k, v = _rand_bf16((L, Hkv, 21, D), 1), _rand_bf16((L, Hkv, 21, D), 2, scale=3.0)
    k[0, 0, 6, 3] = 0x7F80                       # no e4m3 value: stored as the NaN code; its rotation partner must survive delta 0
    a = O.OracleLibrary(L, Hq, Hkv, D, page_size=P, rope_mode=rope_mode, rope_base=1e4, n_pages=128)
    b = O.OracleLibrary(L, Hq, Hkv, D, page_size=P, rope_mode=rope_mode, rope_base=1e4, n_pages=128)
    sa = a.segment_register_fp8(k, v, 300)
    sg = a.segments[sa]
    assert sg.fmt == O.FMT_FP8_E4M3 and sg.k.dtype == np.uint8 and sg.k.shape == k.shape and sg.k_exp.shape == k.shape[:3]
    kd = O.f64_to_bf16(O.fp8_dequantize_rows(sg.k, sg.k_exp))
    vd = O.f64_to_bf16(O.fp8_dequantize_rows(sg.v, sg.v_exp))
    dq = O.fp8_dequantize_rows(sg.k, sg.k_exp)
    assert np.array_equal(np.isnan(dq), np.isnan(O.bf16_to_f64(kd))) and np.isnan(dq).sum() == 1
    assert np.array_equal(O.bf16_to_f64(kd)[~np.isnan(dq)], dq[~np.isnan(dq)])           # exact, not merely close
    sb = b.segment_register(kd, vd, 300)
    plan = lambda s: [O.Plan(0, [O.PlanEntry(s, 2, 9, 0), O.PlanEntry(s, 0, 21, 12), O.PlanEntry(s, 5, 4, 302 + 3)], [O.Hole(9, 3)], 0)]
    a.stitch(plan(sa))
    b.stitch(plan(sb))
    ta, tb = a.tasks[0], b.tasks[0]
    assert ta.deltas == tb.deltas and 0 in [ta.deltas[2]]                # the third entry is an identity graft (delta 0)
    nan = (tb.k & 0x7FFF) > 0x7F80
    assert np.array_equal(nan, (ta.k & 0x7FFF) > 0x7F80) and nan.sum() >= 3
    assert np.array_equal(ta.k[~nan], tb.k[~nan]) and np.array_equal(ta.v, tb.v) and np.array_equal(ta.filled, tb.filled)
    assert (nan[:, :, 305:309].sum() == 1) or rope_mode == 0    # the identity graft keeps the NaN to itself
    # and the stored bytes are half of bf16's (+ one exponent per row)
    assert sg.k.nbytes * 2 == k.nbytes


def test_fp8_deep_subnormal_rows_round_once():
    """rows so small that the scale clamps at 2^-127: code * 2^e can fall below bf16's smallest subnormal 2^-133;
    V is then rounded (RNE) to bf16 and K is rounded once after the rotation."""
    tiny = np.asarray([[0x0001, 0x0002, 0x0005, 0x0040, 0x8003, 0x0000, 0x0010, 0x0020]], np.uint16)   # bf16 subnormals
    codes, ex = O.fp8_quantize_rows(tiny)
    assert ex[0] == -127
    dq = O.fp8_dequantize_rows(codes, ex)
    x = O.bf16_to_f64(tiny)
    assert np.all(np.abs(dq - x) <= 2.0 ** -10 * 2.0 ** -127 + np.abs(x) * 2.0 ** -4)
    lib = O.OracleLibrary(1, 1, 1, 8, page_size=4, n_pages=4)
    s = lib.segment_register_fp8(tiny[None, None], tiny[None, None], 0)
    lib.stitch([O.Plan(0, [O.PlanEntry(s, 0, 1, 0)])])
    assert np.array_equal(lib.tasks[0].v[0, 0], O.f64_to_bf16(dq))
    assert np.array_equal(lib.tasks[0].k[0, 0], O.f64_to_bf16(dq))       # delta 0: cos 0 = 1, sin 0 = 0 exactly


def test_rotation_by_zero_is_the_identity_on_every_bit_pattern():
    """P2 / 8(c).1: delta = 0 leaves every bf16 pattern alone -- infinities, NaN payloads, -0, subnormals -- for a
    scalar delta and for the rows of a per-row delta array that are 0; the other rows are rotated."""
    th = O.rope_inv_freq(16, 1e4)
    allbits = np.arange(65536, dtype=np.uint16).reshape(-1, 16)
    for mode in (O.ROPE_HALF_SPLIT, O.ROPE_INTERLEAVED):
        assert np.array_equal(O.rope_shift_bf16(allbits, 0, th, mode), allbits)
        deltas = np.where(np.arange(allbits.shape[0]) % 2 == 0, 0, 5)
        got = O.rope_shift_bf16(allbits, deltas, th, mode)
        assert np.array_equal(got[0::2], allbits[0::2])
        assert np.array_equal(got[1::2], O.rope_shift_bf16(allbits[1::2], 5, th, mode))
    # and a non-zero rotation propagates specials as IEEE arithmetic does: inf stays inf (sign by the cos / sin), NaN stays NaN
    row = np.zeros((1, 16), np.uint16)
    row[0, 2] = 0x7F80                                   # +inf in the low half, partner (element 10) = 0
    out = O.bf16_to_f64(O.rope_shift_bf16(row, 3, th))
    c, s = np.cos(3 * th[2]), np.sin(3 * th[2])
    assert out[0, 2] == np.copysign(np.inf, c) and out[0, 10] == np.copysign(np.inf, s)
    row[0, 10] = 0x7FC0
    assert np.isnan(O.bf16_to_f64(O.rope_shift_bf16(row, 3, th))[0, [2, 10]]).all()


def test_stitch_with_prefetch_changes_residency_only():
    L, Hq, Hkv, D = 1, 2, 1, 16
    libs = []
    for prefetch in (False, True):
        lib = O.OracleLibrary(L, Hq, Hkv, D, page_size=4, n_pages=32)
        for i in range(3):
            lib.segment_register(_rand_bf16((L, Hkv, 9, D), i), _rand_bf16((L, Hkv, 9, D), 10 + i), 5 * i)
        lib.segment_offload(0)
        lib.segment_offload(2)
        lib.stitch([O.Plan(0, [O.PlanEntry(0, 0, 9, 0), O.PlanEntry(1, 2, 5, 9)])], prefetch=prefetch)
        libs.append(lib)
    a, b = libs
    assert np.array_equal(a.tasks[0].k, b.tasks[0].k) and np.array_equal(a.tasks[0].v, b.tasks[0].v)
    assert a.tasks[0].page_table == b.tasks[0].page_table
    assert [a.segment_info(i)[2] for i in range(3)] == [False, True, False]
    assert [b.segment_info(i)[2] for i in range(3)] == [True, True, False]      # only the segments the plan names come back
