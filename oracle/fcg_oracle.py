"""CPU oracle for FCGRAFT KV-cache grafting.  TEST INFRASTRUCTURE ONLY.

This file is the plain, slow, obviously-correct statement of what the hot path
computes.  It is imported only by ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py``.  The product
(``paper_2606_13097_b200``) never imports it, and it never imports the product:
the two share no code, no tables, no helpers.

Everything is numpy, fp64, one rounding (fp64 -> bf16, round-to-nearest-even)
at the very end of each step that stores bf16.  K/V/q are carried around as
``uint16`` arrays holding bf16 bit patterns, so "bit-exact" means integer
equality of those arrays.

What the paper fixes and what it leaves open (``PAPER.md`` = /root/reference/PAPER.md,
not needed at run time; DESIGN.md "Readings" lists every choice R1..R26):

* segment library  = the KV half of the two-tier code cache H=(I,C), Eq. (2),
  PAPER.md:66-79: per function a K/V state that can be re-injected "without
  being tied to fixed prefix positions".
* cache-stitching  = Eq. (4): cached KV states are
  "concatenated and injected ... as additional context", each module
  "preserving its internal token order during composition".
* cache-patching   = Eq. (6): prefix KV reused, only
  the middle span recomputed, suffix kept.
* The paper never says how positions are reconciled; BASELINE.json's north_star
  fixes it: keys are re-rotated by the integer position delta (RoPE group law),
  values are untouched (R1).  Pair layout: HF half-split (R2).

NEXT rows of SURVEY.md 8(f) stated here as well: interleaved RoPE pairs
(rope_mode 2), ``task_shift`` (re-graft of the kept suffix after a patch of
another length, Eq. 6), ``segment_extract`` (`update` of Alg. 1B),
residency flags (Eq. 3), ``patch_rope``, the locality score of Eq. 3 / 8-10 (``LocalityScore``), fp8 (e4m3)
segment storage (``segment_register_fp8``, R26) and appends beyond the reserved capacity (``check_patch``, R25).

Pinned by tests/test_oracle_pins.py (group law, identity, synthetic one-layer
model, brute-force attention, closed forms, torch SDPA special case, complex
multiplication for both pair layouts, a hand-computed paging example for
task_shift, extract/stitch round trips ...) and tests/test_oracle_pins_r2.py (hand-computed
page tables of a growing task; all 256 e4m3 codes against torch's float8 type, nearest-code
brute force, a hand-worked quantised row).  No function here is "parity unpinned".
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

# ----------------------------------------------------------------------------
# status codes (values are part of the C ABI contract in include/fcg.h; the
# oracle restates them so that plan-rejection behaviour can be compared)
# ----------------------------------------------------------------------------
FCG_OK = 0
FCG_ERR_INVALID_ARG = -1
FCG_ERR_BAD_SEGMENT = -2
FCG_ERR_RANGE = -3
FCG_ERR_OVERLAP = -4
FCG_ERR_UNFILLED = -5
FCG_ERR_OUT_OF_PAGES = -6
FCG_ERR_OUT_OF_ARENA = -7
FCG_ERR_CUDA = -8
FCG_ERR_BAD_TASK = -9


class OracleError(Exception):
    def __init__(self, status: int, msg: str):
        super().__init__(f"status {status}: {msg}")
        self.status = status


# ----------------------------------------------------------------------------
# 1. bf16 <-> fp64                                   (DESIGN R4)
# ----------------------------------------------------------------------------
def bf16_to_f64(bits) -> np.ndarray:
    """bf16 bit patterns (uint16) -> float64, exact (bf16 is a prefix of fp32)."""
    b = np.ascontiguousarray(bits, dtype=np.uint16)
    with np.errstate(invalid="ignore"):            # signalling-NaN patterns widen to NaN, quietly
        return (b.astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)


def f64_to_bf16(x) -> np.ndarray:
    """float64 -> bf16 bit patterns, ONE direct round-to-nearest-even.

    bf16 has 8 significant bits and fp32's exponent range.  For x in
    [2^E, 2^(E+1)) with E >= -126 the bf16 grid has spacing q = 2^(E-7); below
    2^-126 (subnormals) the spacing stays 2^-133.  x/q is exact (power of two),
    np.rint rounds half to even, so r = rint(x/q)*q is the correctly rounded
    bf16 value; it is exactly representable in fp32, whose top 16 bits are the
    answer.  |r| >= 2^128 becomes inf; NaN stays NaN.  Never goes through fp32
    rounding of the *unrounded* value (no double rounding).
    """
    x = np.asarray(x, dtype=np.float64)
    _, e = np.frexp(x)                     # |x| = m * 2^e, m in [0.5, 1)  =>  floor(log2|x|) = e - 1
    E = np.maximum(e - 1, -126)
    q = np.ldexp(1.0, E - 7)
    with np.errstate(over="ignore", invalid="ignore"):
        r = np.rint(x / q) * q
        r32 = r.astype(np.float32)         # exact unless |r| >= 2^128 -> inf (what bf16 RNE overflow gives)
    return (r32.view(np.uint32) >> np.uint32(16)).astype(np.uint16)


# ----------------------------------------------------------------------------
# 2. RoPE delta rotation                              (DESIGN R1-R4)
# ----------------------------------------------------------------------------
def rope_inv_freq(head_dim: int, base: float) -> np.ndarray:
    """theta_j = base^(-2j/D), j in [0, D/2), fp64 pow."""
    j = np.arange(head_dim // 2, dtype=np.float64)
    return np.power(np.float64(base), -2.0 * j / np.float64(head_dim))


ROPE_NONE, ROPE_HALF_SPLIT, ROPE_INTERLEAVED = 0, 1, 2


def rope_rotate_f64(x: np.ndarray, delta, inv_freq: np.ndarray, rope_mode: int = ROPE_HALF_SPLIT) -> np.ndarray:
    """Rotate x[..., D] (fp64) by the position delta; result fp64, NOT rounded.

    Pair j is (a, b) = (x[j], x[j + D/2]) for half-split pairs (HF convention,
    DESIGN R2) or (x[2j], x[2j + 1]) for interleaved pairs (GPT-J / original
    RoFormer convention):
        phi_j  = delta * theta_j
        a' = a cos(phi_j) - b sin(phi_j)
        b' = b cos(phi_j) + a sin(phi_j)
    ``delta`` is an integer, or an array broadcastable against x[..., :1]
    (one delta per row).
    """
    x = np.asarray(x, dtype=np.float64)
    D = x.shape[-1]
    half = D // 2
    phi = np.asarray(delta, dtype=np.float64)[..., None] * inv_freq     # scalar delta -> [D/2]; per-row -> [..., D/2]
    c, s = np.cos(phi), np.sin(phi)
    out = np.empty_like(x)
    with np.errstate(invalid="ignore"):            # inf - inf, inf * 0 are NaN, quietly (IEEE special values propagate)
        if rope_mode == ROPE_HALF_SPLIT:
            a, b = x[..., :half], x[..., half:]
            out[..., :half] = a * c - b * s
            out[..., half:] = b * c + a * s
        elif rope_mode == ROPE_INTERLEAVED:
            a, b = x[..., 0::2], x[..., 1::2]
            out[..., 0::2] = a * c - b * s
            out[..., 1::2] = b * c + a * s
        else:
            raise OracleError(FCG_ERR_INVALID_ARG, "rope_mode must be half-split (1) or interleaved (2) to rotate")
    return out


def rope_shift_bf16(k_bits: np.ndarray, delta, inv_freq: np.ndarray, rope_mode: int = ROPE_HALF_SPLIT) -> np.ndarray:
    """bf16 keys -> bf16 keys rotated by ``delta``: fp64 arithmetic, one RNE.

    delta == 0 is the identity ON THE BITS ("grafted with delta 0 -> K bit-identical to the source";
    8(c).1: "+-inf / NaN propagate"): evaluating a cos 0 - b sin 0 literally would turn an infinite a or b into NaN
    through inf * 0 and would canonicalise NaN payloads, which a rotation by nothing must not do.
    """
    k_bits = np.asarray(k_bits, dtype=np.uint16)
    out = f64_to_bf16(rope_rotate_f64(bf16_to_f64(k_bits), delta, inv_freq, rope_mode))
    same = np.broadcast_to(np.asarray(delta)[..., None] == 0, k_bits.shape)
    return np.where(same, k_bits, out)


# ----------------------------------------------------------------------------
# 2b. fp8 (e4m3) segment storage                     (DESIGN R26)
# ----------------------------------------------------------------------------
# OCP 8-bit float E4M3 ("e4m3fn"): 1 sign, 4 exponent bits (bias 7), 3 mantissa bits; no infinities; the only NaN
# is S.1111.111; largest finite value 1.75 * 2^8 = 448; subnormals m/8 * 2^-6.  A stored row (the D elements of one
# (layer, kv head, token)) shares one power-of-two scale 2^e (an E8M0 exponent, as in the OCP MX formats), so that
# de-quantisation code * 2^e is exact and the shifted key is still ONE rounding away from the exact rotation.
E4M3_MAX = 448.0
FMT_BF16, FMT_FP8_E4M3 = 0, 1


def e4m3_to_f64(codes) -> np.ndarray:
    """e4m3 codes (uint8) -> float64, exact."""
    c = np.ascontiguousarray(codes, dtype=np.uint8).astype(np.int64)
    sign = np.where(c & 0x80, -1.0, 1.0)
    e, m = (c >> 3) & 0xF, (c & 7).astype(np.float64)
    val = np.where(e == 0, np.ldexp(m / 8.0, -6), np.ldexp(1.0 + m / 8.0, e - 7))
    return np.where((e == 15) & (m == 7), np.nan, sign * val)


def f64_to_e4m3(x) -> np.ndarray:
    """float64 -> e4m3 code, round-to-nearest-even on the e4m3 grid, finite overflow saturates to +-448
    ("satfinite"); NaN and +-inf have no e4m3 value and become the NaN code 0x7F."""
    x = np.asarray(x, dtype=np.float64)
    a = np.abs(x)
    finite = np.isfinite(x)
    a = np.where(finite, a, 0.0)
    _, ex = np.frexp(a)                                   # a = m * 2^ex, m in [0.5, 1)
    E = np.maximum(ex - 1, -6)                            # exponent of the binade; subnormals share 2^-6's quantum
    q = np.ldexp(1.0, E - 3)                              # grid spacing: 3 mantissa bits
    r = np.minimum(np.rint(a / q) * q, E4M3_MAX)          # a / q is exact; rint = half to even; then saturate
    _, rex = np.frexp(r)
    rE = rex - 1
    normal = r >= 2.0 ** -6
    e_bits = np.where(normal, rE + 7, 0).astype(np.int64)
    m_bits = np.where(normal, np.rint((np.ldexp(r, -rE) - 1.0) * 8.0), np.rint(np.ldexp(r, 9))).astype(np.int64)
    code = (e_bits << 3) | m_bits
    code = np.where(np.signbit(x), code | 0x80, code)
    return np.where(finite, code, 0x7F).astype(np.uint8)


def fp8_row_exponent(x) -> np.ndarray:
    """Per-row scale exponent e for rows x[..., D] (fp64): the smallest integer with amax <= 448 * 2^e, clamped to
    the E8M0 range [-127, 127]; amax is taken over the finite elements; an all-zero row gets e = 0.  Integer
    arithmetic on the binary exponent (448 = 0.875 * 2^9), no logarithm."""
    x = np.asarray(x, dtype=np.float64)
    amax = np.max(np.where(np.isfinite(x), np.abs(x), 0.0), axis=-1)
    m, ex = np.frexp(amax)
    e = np.where(m <= 0.875, ex - 9, ex - 8)
    e = np.where(amax == 0.0, 0, e)
    return np.clip(e, -127, 127).astype(np.int32)


def fp8_quantize_rows(bits):
    """bf16 rows [..., D] -> (e4m3 codes uint8 [..., D], scale exponents int32 [...]): code = e4m3(x * 2^-e)."""
    x = bf16_to_f64(bits)
    e = fp8_row_exponent(x)
    return f64_to_e4m3(np.ldexp(x, -e[..., None])), e


def fp8_dequantize_rows(codes, exps) -> np.ndarray:
    """(codes [..., D], exponents [...]) -> float64 [..., D] = value(code) * 2^e, exact."""
    return np.ldexp(e4m3_to_f64(codes), np.asarray(exps, dtype=np.int32)[..., None])


# ----------------------------------------------------------------------------
# 3. page pool                                         (DESIGN R9)
# ----------------------------------------------------------------------------
class PagePool:
    """Deterministic LIFO page allocator: a fresh pool hands out 0, 1, 2, ...

    ``release`` pushes pages back so that the *next* allocation returns them in
    the order they are listed (i.e. a released task's pages are re-issued in
    ascending logical order).
    """

    def __init__(self, n_pages: int):
        self.n_pages = int(n_pages)
        self._stack = list(range(self.n_pages - 1, -1, -1))   # pop() -> 0, 1, 2, ...

    def available(self) -> int:
        return len(self._stack)

    def allocate(self, n: int) -> list[int]:
        if n > len(self._stack):
            raise OracleError(FCG_ERR_OUT_OF_PAGES, f"need {n} pages, {len(self._stack)} free")
        return [self._stack.pop() for _ in range(n)]

    def release(self, pages: list[int]) -> None:
        for p in reversed(pages):
            self._stack.append(p)


# ----------------------------------------------------------------------------
# 4. library / plans / tasks
# ----------------------------------------------------------------------------
@dataclass
class Segment:
    k: np.ndarray            # [L][Hkv][n][D] uint16 (bf16 bits), owned copy
    v: np.ndarray
    n_tokens: int
    orig_start: int          # position at which token 0's key was RoPE-encoded
    resident: bool = True    # False: offloaded to the host tier (Eq. 3); the bits are the same wherever they live
    fmt: int = 0             # FMT_BF16: k, v hold bf16 bits; FMT_FP8_E4M3: k, v hold e4m3 codes (uint8) and
    k_exp: np.ndarray = None  # k_exp, v_exp [L][Hkv][n] the per-row power-of-two scale exponents (R26)
    v_exp: np.ndarray = None


@dataclass
class PlanEntry:
    seg_id: int
    src_begin: int
    n_tokens: int
    dst_offset: int


@dataclass
class Hole:
    begin: int
    n_tokens: int


@dataclass
class Plan:
    task_id: int
    entries: list
    holes: list = field(default_factory=list)
    capacity_tokens: int = 0       # 0 -> max end of entries/holes


@dataclass
class Task:
    page_table: list          # logical page -> physical page id
    capacity: int
    n_tokens: int             # T: max filled-or-declared end
    filled: np.ndarray        # bool[capacity]
    k: np.ndarray             # logical cache [L][Hkv][capacity][D] uint16
    v: np.ndarray
    deltas: list              # per entry, for inspection
    spans: list = field(default_factory=list)   # (dst_offset, n_tokens) of every stitched entry, in plan order


class OracleLibrary:
    """Plain restatement of the library state machine behind the C ABI."""

    def __init__(self, n_layers, n_q_heads, n_kv_heads, head_dim, page_size=16,
                 rope_mode=1, rope_base=1e4, inv_freq=None, max_segments=1 << 16,
                 max_tasks=1 << 16, n_pages=1 << 20, max_task_tokens=1 << 30):
        if head_dim % 8 or head_dim <= 0 or n_q_heads % n_kv_heads or page_size <= 0:
            raise OracleError(FCG_ERR_INVALID_ARG, "bad geometry")
        self.L, self.Hq, self.Hkv, self.D, self.P = n_layers, n_q_heads, n_kv_heads, head_dim, page_size
        self.G = n_q_heads // n_kv_heads
        self.rope_mode = rope_mode
        self.inv_freq = (np.asarray(inv_freq, dtype=np.float64) if inv_freq is not None
                         else rope_inv_freq(head_dim, rope_base))
        self.max_segments, self.max_tasks, self.max_task_tokens = max_segments, max_tasks, max_task_tokens
        self.pool = PagePool(n_pages)
        self.segments: dict[int, Segment] = {}
        self.tasks: dict[int, Task] = {}
        self._next_seg = 0

    # -- S1 ------------------------------------------------------------------
    def segment_register(self, k_bits, v_bits, orig_start: int) -> int:
        """Keep the K/V bits, orig_start and n."""
        k = np.array(k_bits, dtype=np.uint16, copy=True)
        v = np.array(v_bits, dtype=np.uint16, copy=True)
        if k.shape != v.shape or k.ndim != 4 or k.shape[0] != self.L or k.shape[1] != self.Hkv \
                or k.shape[3] != self.D or k.shape[2] <= 0 or orig_start < 0:
            raise OracleError(FCG_ERR_INVALID_ARG, "segment shape must be [L][Hkv][n][D], n > 0, orig_start >= 0")
        # lowest free id (ids of released segments are reused, smallest first)
        sid = 0
        while sid in self.segments:
            sid += 1
        if sid >= self.max_segments:
            raise OracleError(FCG_ERR_OUT_OF_ARENA, "segment table full")
        self.segments[sid] = Segment(k, v, k.shape[2], int(orig_start))
        return sid

    def segment_register_fp8(self, k_bits, v_bits, orig_start: int) -> int:
        """S1 with fp8 storage (DESIGN R26): the bf16 K/V handed in are quantised row by row to
        e4m3 codes with a power-of-two row scale; the library keeps codes + exponents (half the bytes of bf16)."""
        sid = self.segment_register(k_bits, v_bits, orig_start)      # shape checks and id rule as for bf16
        sg = self.segments[sid]
        sg.k, sg.k_exp = fp8_quantize_rows(sg.k)
        sg.v, sg.v_exp = fp8_quantize_rows(sg.v)
        sg.fmt = FMT_FP8_E4M3
        return sid

    def segment_release(self, seg_id: int) -> None:
        if seg_id not in self.segments:
            raise OracleError(FCG_ERR_BAD_SEGMENT, f"unknown segment {seg_id}")
        del self.segments[seg_id]

    # -- NEXT-3: two-tier residency (Eq. 3, Table 19) ----------------
    def segment_offload(self, seg_id: int) -> None:
        """Low-scored entries "are offloaded to DRAM".  Which entries is the caller's policy (the
        locality score of Eq. 3 is not on the path); the library only moves the bits.  Values do not change:
        stitching from an offloaded segment gives the same cache.  Idempotent."""
        if seg_id not in self.segments:
            raise OracleError(FCG_ERR_BAD_SEGMENT, f"unknown segment {seg_id}")
        self.segments[seg_id].resident = False

    def segment_prefetch(self, seg_id: int) -> None:
        """CPU -> GPU reload "only when a required function cache is not resident".  Idempotent."""
        if seg_id not in self.segments:
            raise OracleError(FCG_ERR_BAD_SEGMENT, f"unknown segment {seg_id}")
        self.segments[seg_id].resident = True

    def segment_info(self, seg_id: int):
        """(n_tokens, orig_start, resident)"""
        if seg_id not in self.segments:
            raise OracleError(FCG_ERR_BAD_SEGMENT, f"unknown segment {seg_id}")
        sg = self.segments[seg_id]
        return sg.n_tokens, sg.orig_start, sg.resident

    # -- S2 ------------------------------------------------------------------
    def validate_plan(self, plan: Plan):
        """Returns (capacity, T, deltas).  Raises OracleError; changes no state.

        Rules (DESIGN R5-R7): 0 <= src_begin, n > 0,
        src_begin + n <= n_seg, dst_offset >= 0, end <= capacity; entries and
        holes pairwise disjoint; delta_e = dst_offset - orig_start - src_begin.
        """
        if plan.task_id < 0 or plan.task_id >= self.max_tasks:
            raise OracleError(FCG_ERR_BAD_TASK, "task id out of range")
        if plan.task_id in self.tasks:
            raise OracleError(FCG_ERR_BAD_TASK, "task id already live")
        if len(plan.entries) + len(plan.holes) == 0:
            raise OracleError(FCG_ERR_INVALID_ARG, "empty plan")
        spans, deltas = [], []
        for e in plan.entries:
            if e.seg_id not in self.segments:
                raise OracleError(FCG_ERR_BAD_SEGMENT, f"unknown segment {e.seg_id}")
            seg = self.segments[e.seg_id]
            if e.n_tokens <= 0 or e.src_begin < 0 or e.src_begin + e.n_tokens > seg.n_tokens or e.dst_offset < 0:
                raise OracleError(FCG_ERR_RANGE, "entry source/destination range")
            spans.append((e.dst_offset, e.dst_offset + e.n_tokens))
            deltas.append(e.dst_offset - seg.orig_start - e.src_begin)
        for h in plan.holes:
            if h.n_tokens <= 0 or h.begin < 0:
                raise OracleError(FCG_ERR_RANGE, "hole range")
            spans.append((h.begin, h.begin + h.n_tokens))
        T = max(end for _, end in spans)
        capacity = plan.capacity_tokens if plan.capacity_tokens > 0 else T
        if T > capacity:
            raise OracleError(FCG_ERR_RANGE, "plan exceeds capacity_tokens")
        if capacity > self.max_task_tokens:
            raise OracleError(FCG_ERR_RANGE, "capacity exceeds max_task_tokens")
        srt = sorted(spans)
        for (b0, e0), (b1, e1) in zip(srt, srt[1:]):
            if b1 < e0:
                raise OracleError(FCG_ERR_OVERLAP, "entries/holes overlap")
        return capacity, T, deltas

    # -- S2 + S3 -------------------------------------------------------------
    def stitch(self, plans: list, prefetch: bool = False) -> None:
        """Build page tables and gather + RoPE-shift (Eq. 4).

        ``prefetch`` (reloads "only when a required function cache is not
        resident"): offloaded segments named by the plans come back to the device tier as part of the call; the
        stitched cache is the same either way -- only the residency flags differ afterwards.

        All plans are validated and all pages reserved before any state
        changes (allocate-then-commit): a failing batch leaves the library as
        it was.
        """
        checked = []
        seen = set()
        need = 0
        for plan in plans:
            if plan.task_id in seen:
                raise OracleError(FCG_ERR_BAD_TASK, "task id repeated in batch")
            seen.add(plan.task_id)
            cap, T, deltas = self.validate_plan(plan)
            n_pg = -(-cap // self.P)
            need += n_pg
            checked.append((plan, cap, T, deltas, n_pg))
        if need > self.pool.available():
            raise OracleError(FCG_ERR_OUT_OF_PAGES, f"need {need} pages, {self.pool.available()} free")
        if prefetch:
            for plan, *_ in checked:
                for e in plan.entries:
                    self.segments[e.seg_id].resident = True
        for plan, cap, T, deltas, n_pg in checked:
            table = self.pool.allocate(n_pg)           # plans in array order, pages in ascending logical order
            kc = np.zeros((self.L, self.Hkv, cap, self.D), np.uint16)
            vc = np.zeros_like(kc)
            filled = np.zeros(cap, bool)
            for e, delta in zip(plan.entries, deltas):
                seg = self.segments[e.seg_id]
                src = slice(e.src_begin, e.src_begin + e.n_tokens)
                dst = slice(e.dst_offset, e.dst_offset + e.n_tokens)
                if seg.fmt == FMT_FP8_E4M3:
                    # R26: de-quantise (exact), rotate in fp64, ONE rounding to bf16; V: de-quantise, round to bf16
                    # (exact whenever code * 2^e is a bf16 value, i.e. everywhere but the deepest subnormals)
                    kf = fp8_dequantize_rows(seg.k[:, :, src], seg.k_exp[:, :, src])
                    if self.rope_mode != 0 and delta != 0:         # delta 0 is the identity (P2), also for a NaN partner
                        kf = rope_rotate_f64(kf, delta, self.inv_freq, self.rope_mode)
                    kc[:, :, dst] = f64_to_bf16(kf)
                    vc[:, :, dst] = f64_to_bf16(fp8_dequantize_rows(seg.v[:, :, src], seg.v_exp[:, :, src]))
                    filled[dst] = True
                    continue
                if self.rope_mode == 0:
                    kc[:, :, dst] = seg.k[:, :, src]                       # pure gather
                else:
                    kc[:, :, dst] = rope_shift_bf16(seg.k[:, :, src], delta, self.inv_freq, self.rope_mode)
                vc[:, :, dst] = seg.v[:, :, src]                           # V: bit copy
                filled[dst] = True
            self.tasks[plan.task_id] = Task(table, cap, T, filled, kc, vc, deltas,
                                            [(e.dst_offset, e.n_tokens) for e in plan.entries])

    # -- S4 + S5/S6 ----------------------------------------------------------
    def check_patch(self, task_id: int, positions) -> int:
        """Validates a patch; changes no state.  Returns the number of pages the patch has to add.

        SURVEY 8(c).5 / DESIGN R25: positions beyond the task's current capacity APPEND -- the task grows to
        capacity' = positions[-1] + 1 (never beyond max_task_tokens: RANGE) and takes the logical pages
        ceil(capacity / P) .. ceil(capacity' / P) - 1 from the pool on demand (OUT_OF_PAGES if it cannot supply
        them).  Positions between the old and the new capacity are unfilled until somebody writes them, so the
        rule "every x <= positions[-1] is filled by earlier work or by this call" (R6) covers growth as well.
        """
        if task_id not in self.tasks:
            raise OracleError(FCG_ERR_BAD_TASK, f"unknown task {task_id}")
        t = self.tasks[task_id]
        pos = np.asarray(positions, dtype=np.int64)
        if pos.ndim != 1 or pos.size == 0:
            raise OracleError(FCG_ERR_INVALID_ARG, "positions must be a non-empty 1-d array")
        if np.any(np.diff(pos) <= 0):
            raise OracleError(FCG_ERR_INVALID_ARG, "positions must be strictly increasing")
        if pos[0] < 0 or pos[-1] >= self.max_task_tokens:
            raise OracleError(FCG_ERR_RANGE, "position outside [0, max_task_tokens)")
        cap = max(t.capacity, int(pos[-1]) + 1)
        f = np.zeros(cap, bool)
        f[: t.capacity] = t.filled
        f[pos] = True
        if not np.all(f[: pos[-1] + 1]):
            raise OracleError(FCG_ERR_UNFILLED, "a patch query would attend over an unfilled position")
        need = -(-cap // self.P) - len(t.page_table)
        if need > self.pool.available():
            raise OracleError(FCG_ERR_OUT_OF_PAGES, f"need {need} pages to grow, {self.pool.available()} free")
        return max(need, 0)

    def _grow(self, task_id: int, capacity: int, n_new_pages: int) -> None:
        """Append pages (ascending logical order, from the LIFO pool) and extend the logical cache (R25)."""
        t = self.tasks[task_id]
        t.page_table.extend(self.pool.allocate(n_new_pages))
        if capacity > t.capacity:
            extra = capacity - t.capacity
            pad = np.zeros((self.L, self.Hkv, extra, self.D), np.uint16)
            t.k = np.concatenate([t.k, pad], axis=2)
            t.v = np.concatenate([t.v, pad.copy()], axis=2)
            t.filled = np.concatenate([t.filled, np.zeros(extra, bool)])
            t.capacity = capacity

    def patch_rope(self, task_id: int, layer_begin: int, q_bits, k_bits, v_bits, positions) -> np.ndarray:
        """patch() for callers that hold the projections BEFORE position encoding (DESIGN R13
        variant): token i's query and key are first rotated to its absolute position p_i by the library's RoPE
        (theta_j and pair layout of the configuration), each rounded once to bf16 -- what a model's own RoPE would
        have handed to patch() -- then scattered / attended exactly as in patch().  rope_mode NONE: identical to patch().
        """
        pos = np.asarray(positions, dtype=np.int64)
        q_bits = np.asarray(q_bits, np.uint16)
        k_bits = np.asarray(k_bits, np.uint16)
        if self.rope_mode != ROPE_NONE and pos.ndim == 1 and q_bits.ndim == 4 and k_bits.ndim == 4 \
                and q_bits.shape[1] == pos.size and k_bits.shape[1] == pos.size:
            per_row = pos[None, :, None]                                   # one delta per (layer, token, head) row
            q_bits = rope_shift_bf16(q_bits, np.broadcast_to(per_row, q_bits.shape[:3]), self.inv_freq, self.rope_mode)
            k_bits = rope_shift_bf16(k_bits, np.broadcast_to(per_row, k_bits.shape[:3]), self.inv_freq, self.rope_mode)
        return self.patch(task_id, layer_begin, q_bits, k_bits, v_bits, positions)

    def patch(self, task_id: int, layer_begin: int, q_bits, k_bits, v_bits, positions) -> np.ndarray:
        """Scatter then causal patch attention (Eq. 6).

        q_bits [nl][n][Hq][D], k_bits/v_bits [nl][n][Hkv][D] (uint16 bf16 bits,
        already position-encoded by the caller, DESIGN R13).  Returns the
        attention output as float64 [nl][n][Hq][D], NOT rounded.
        Query i at position p_i sees cache positions x <= p_i (DESIGN R12).
        Positions at or beyond the current capacity append: the task grows page by page (check_patch, R25).
        """
        n_new_pages = self.check_patch(task_id, positions)
        pos = np.asarray(positions, dtype=np.int64)
        q_bits = np.asarray(q_bits, np.uint16)
        k_bits = np.asarray(k_bits, np.uint16)
        v_bits = np.asarray(v_bits, np.uint16)
        nl, n = q_bits.shape[0], pos.size
        if layer_begin < 0 or nl <= 0 or layer_begin + nl > self.L \
                or q_bits.shape != (nl, n, self.Hq, self.D) or k_bits.shape != (nl, n, self.Hkv, self.D) \
                or v_bits.shape != k_bits.shape:
            raise OracleError(FCG_ERR_INVALID_ARG, "patch tensor shapes / layer range")
        self._grow(task_id, max(self.tasks[task_id].capacity, int(pos[-1]) + 1), n_new_pages)   # R25: append on demand
        t = self.tasks[task_id]
        out = np.empty((nl, n, self.Hq, self.D), np.float64)
        for li in range(nl):
            layer = layer_begin + li
            # S4: scatter (bit copy) -- happens before this layer's attention
            t.k[layer][:, pos, :] = np.transpose(k_bits[li], (1, 0, 2))
            t.v[layer][:, pos, :] = np.transpose(v_bits[li], (1, 0, 2))
            out[li] = patch_attention(t.k[layer], t.v[layer], q_bits[li], pos, self.G)
        t.filled[pos] = True
        t.n_tokens = max(t.n_tokens, int(pos[-1]) + 1)
        return out

    # -- NEXT-1: length-changing patch = re-graft of the suffix ------------------
    def task_shift(self, task_id: int, src_begin: int, n_tokens: int, dst_begin: int) -> None:
        """Move cache positions [src_begin, src_begin+n) of a live task to [dst_begin, dst_begin+n).

        Eq. (6): after the erroneous span x_err is replaced by an x_mid of another
        length, the kept suffix sits delta = dst_begin - src_begin positions further; its keys are
        re-rotated by delta (same rule as stitching, DESIGN R1), values are bit-copied (DESIGN R15,
        SURVEY 8(f) NEXT-1).  Source positions become unfilled, destination positions filled (a
        destination position that was filled is overwritten).  T never shrinks.

        Paging ("copy-on-shift", so that no page is read and written in the same pass): every logical
        page touched by the destination range gets a fresh physical page from the pool (ascending
        logical order); slots of those pages outside the destination range keep their old contents;
        the old physical pages go back to the pool by the rule of task_release.  delta == 0 is a no-op.
        The source must lie inside the capacity; the destination may reach beyond it (up to max_task_tokens): the
        task then grows as for an appending patch (R25).
        """
        if task_id not in self.tasks:
            raise OracleError(FCG_ERR_BAD_TASK, f"unknown task {task_id}")
        t = self.tasks[task_id]
        if n_tokens <= 0 or src_begin < 0 or dst_begin < 0 or src_begin + n_tokens > t.capacity \
                or dst_begin + n_tokens > self.max_task_tokens:
            raise OracleError(FCG_ERR_RANGE, "shift source outside the capacity / destination outside max_task_tokens")
        src = slice(src_begin, src_begin + n_tokens)
        dst = slice(dst_begin, dst_begin + n_tokens)
        if not np.all(t.filled[src]):
            raise OracleError(FCG_ERR_UNFILLED, "shift source holds an unfilled position")
        delta = dst_begin - src_begin
        if delta == 0:
            return
        # R25: a destination beyond the capacity appends.  Every logical page that receives a new physical page --
        # the gap pages between the end of the table and the destination, then the destination's pages -- is served
        # in ascending logical order; destination pages that already existed give their old page back.
        n_old = len(t.page_table)
        lp0, lp1 = dst_begin // self.P, (dst_begin + n_tokens - 1) // self.P
        first_new = min(lp0, n_old)
        new_pages = self.pool.allocate(lp1 - first_new + 1)     # raises OUT_OF_PAGES before any change
        k_src = t.k[:, :, src].copy()
        v_src = t.v[:, :, src].copy()
        self._grow(task_id, max(t.capacity, dst_begin + n_tokens), 0)
        if self.rope_mode == ROPE_NONE:
            t.k[:, :, dst] = k_src
        else:
            t.k[:, :, dst] = rope_shift_bf16(k_src, delta, self.inv_freq, self.rope_mode)
        t.v[:, :, dst] = v_src
        t.filled[src] = False
        t.filled[dst] = True
        old_pages = t.page_table[lp0:lp1 + 1]                   # destination pages that existed before
        t.page_table[first_new:lp1 + 1] = new_pages
        self.pool.release(old_pages)
        t.n_tokens = max(t.n_tokens, dst_begin + n_tokens)

    # -- NEXT-2: `update` of Alg. 1B -- cut a function out of a live cache ---------
    def segment_extract(self, task_id: int, begin: int, n_tokens: int, new_orig_start: int) -> int:
        """New library segment from cache positions [begin, begin+n) of a live task (PAPER.md:81, 85:
        `update` inserts the KV state of a newly generated function into the code cache; SURVEY 8(f)
        NEXT-2).  Keys are re-rotated by delta = new_orig_start - begin so that the stored segment is
        encoded as if its first token sat at new_orig_start (begin -> bit copy; 0 -> canonical form);
        values are bit-copied.  Returns the segment id (lowest free id, as segment_register).
        """
        if task_id not in self.tasks:
            raise OracleError(FCG_ERR_BAD_TASK, f"unknown task {task_id}")
        t = self.tasks[task_id]
        if n_tokens <= 0 or begin < 0 or begin + n_tokens > t.capacity:
            raise OracleError(FCG_ERR_RANGE, "extract range outside task capacity")
        if new_orig_start < 0:
            raise OracleError(FCG_ERR_INVALID_ARG, "new_orig_start must be >= 0")
        src = slice(begin, begin + n_tokens)
        if not np.all(t.filled[src]):
            raise OracleError(FCG_ERR_UNFILLED, "extract range holds an unfilled position")
        delta = new_orig_start - begin
        if self.rope_mode == ROPE_NONE or delta == 0:
            k = t.k[:, :, src].copy()
        else:
            k = rope_shift_bf16(t.k[:, :, src], delta, self.inv_freq, self.rope_mode)
        return self.segment_register(k, t.v[:, :, src], new_orig_start)

    def task_boundary_positions(self, task_id: int, width: int) -> list:
        """Positions worth recomputing after a stitch (the boundary-recompute idea of the
        related work the paper positions itself against): the first `width` tokens of every
        stitched entry that does not start at position 0 -- the tokens whose keys / values were computed without
        seeing what now precedes them.  Ascending, without duplicates; the caller recomputes them with the model and
        hands them to patch().  Entries moved later by task_shift are not tracked (the list describes the stitch)."""
        if task_id not in self.tasks:
            raise OracleError(FCG_ERR_BAD_TASK, f"unknown task {task_id}")
        if width <= 0:
            raise OracleError(FCG_ERR_INVALID_ARG, "width must be > 0")
        out = set()
        for (dst, n) in self.tasks[task_id].spans:
            if dst > 0:
                out.update(range(dst, dst + min(width, n)))
        return sorted(out)

    def task_release(self, task_id: int) -> None:
        if task_id not in self.tasks:
            raise OracleError(FCG_ERR_BAD_TASK, f"unknown task {task_id}")
        self.pool.release(self.tasks.pop(task_id).page_table)


# ----------------------------------------------------------------------------
# 5. patch attention, the definition                 (DESIGN R11-R12)
# ----------------------------------------------------------------------------
def patch_attention(k_cache, v_cache, q_bits, positions, group: int) -> np.ndarray:
    """k_cache, v_cache: [Hkv][cap][D] bf16 bits (one layer, logical order);
    q_bits [n][Hq][D]; returns float64 [n][Hq][D].

        g = h // G                      (HF repeat_kv head mapping)
        s_x = q_{i,h} . K[x,g] / sqrt(D)      for x = 0 .. p_i
        o   = sum_x softmax(s)_x V[x,g]
    All in fp64; max-subtraction only for range safety.
    """
    kf = bf16_to_f64(k_cache)
    vf = bf16_to_f64(v_cache)
    qf = bf16_to_f64(q_bits)
    n, Hq, D = qf.shape
    out = np.empty((n, Hq, D), np.float64)
    inv_sqrt_d = 1.0 / math.sqrt(D)
    for i in range(n):
        vis = int(positions[i]) + 1
        for h in range(Hq):
            g = h // group
            s = (kf[g, :vis] @ qf[i, h]) * inv_sqrt_d
            w = np.exp(s - s.max())
            out[i, h] = (w @ vf[g, :vis]) / w.sum()
    return out


# ----------------------------------------------------------------------------
# 6. locality score of the cache management scheme   (Eq. 3, 8, 9, 10)
# ----------------------------------------------------------------------------
class LocalityScore:
    """Bookkeeping behind Eq. (3): which function entries to keep on the GPU and which to offload.

        l(f_k)            = (1 - l_curr) * (alpha * l_freq + beta * sum_j l_asso(f_j | f_k) + gamma * l_sema) + l_curr
        l_freq(f_k)       = count(f_k) / max_j count(f_j)                                   (Eq. 8)
        l_asso(f_j | f_k) = cooccur(f_k, f_j) / count(f_k)                                  (Eq. 9)
        l_sema(f_k)       = PPL(f_k) / max_i PPL(f_i)                                       (Eq. 10)

    Readings (R24): a trace is the sequence of functions one task invoked, in order; count = number of
    invocations over all recorded traces; cooccur(f_k, f_j) = number of times f_j is the NEXT invocation after f_k
    inside a trace ("invoked following f_k"), j != k -- so the sum over j is a conditional likelihood in [0, 1] as
    the paper requires of every component; l_curr = 1 for the functions of the most recently recorded trace; PPL is
    supplied by the caller (it needs the CodeLLM), 0 where unknown.
    """

    def __init__(self):
        self.count = {}
        self.follow = {}        # (k, j) -> times j directly followed k
        self.ppl = {}
        self.last = set()

    def record(self, trace) -> None:
        trace = [int(x) for x in trace]
        for f in trace:
            self.count[f] = self.count.get(f, 0) + 1
        for a, b in zip(trace, trace[1:]):
            if a != b:
                self.follow[(a, b)] = self.follow.get((a, b), 0) + 1
        self.last = set(trace)

    def set_ppl(self, f: int, ppl: float) -> None:
        self.ppl[int(f)] = float(ppl)

    def forget(self, f: int) -> None:
        f = int(f)
        self.count.pop(f, None)
        self.ppl.pop(f, None)
        self.last.discard(f)
        self.follow = {kj: c for kj, c in self.follow.items() if f not in kj}

    def score(self, f: int, alpha: float, beta: float, gamma: float) -> float:
        f = int(f)
        if f in self.last:
            return 1.0
        cnt = self.count.get(f, 0)
        max_cnt = max(self.count.values(), default=0)
        freq = cnt / max_cnt if max_cnt else 0.0
        asso = sum(c for (k, j), c in self.follow.items() if k == f) / cnt if cnt else 0.0
        max_ppl = max(self.ppl.values(), default=0.0)
        sema = self.ppl.get(f, 0.0) / max_ppl if max_ppl > 0 else 0.0
        return alpha * freq + beta * asso + gamma * sema

    def rank(self, ids, alpha: float, beta: float, gamma: float):
        """ids sorted by ascending score (offload candidates first); ties by ascending id."""
        return sorted((int(f) for f in ids), key=lambda f: (self.score(f, alpha, beta, gamma), f))
