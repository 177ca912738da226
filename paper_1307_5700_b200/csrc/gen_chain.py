#!/usr/bin/env python
"""Generates chain_gen.h: the per-slab inner loops of the tiled dedispersion kernels, as inline PTX.

One call of SlabF32<D,T,NOFF>::run / SlabU16<...>::run processes all channels of one staged slab for
one warp:

    for every channel r of the slab (table entry e_r of this warp):
        w[0 .. T+NOFF)  <- shared[sbase + e_r.window_start ...]          (128-bit loads)
        for j < D:  acc[j][i] += w[o_j + i],  i < T                      (o_j = e_r.offset[j], warp-uniform)

Registers cannot be indexed dynamically, so every (j, offset) pair owns a straight-line block of adds and
the blocks are THREADED: block (j, o_j) ends by branching into block (j+1, o_{j+1}).  The dispatch is a short
tree of DIRECT predicated branches on the bits of o_{j+1} (predicates computed at the top of the block, ~2 taken
branches); the PTX `brx.idx` form (SASS LDC jump-table read + BRX; MDSM_GEN_DISPATCH=brx) cost ~90 instead of
~35 warp-cycles per dispatch.  The block of the LAST DM carries a copy of the loop head (next table entry,
window loads, first dispatch) and the whole loop is one asm statement -- nvcc wraps nothing in convergence
barriers (BSSY/BSYNC/BREAK cost ~70 cycles per channel in the r1b profile).  The hot code has to stay inside
the 32 KB L1.5 instruction cache: the integer kernels share one loop head instead of copying it.

Table entry (64 bit):  lo[17:0]  byte offset of the window start inside the stage
                       lo[28+i]  load the optional 16-byte chunk T/4 + i   (i = 0, 1, 2)
                       lo[31]    last channel of the slab for this warp
                       hi        byte j = register offset o_j of DM j

fp32: accumulators and window are packed f32x2 register pairs; an even offset is T/2 FADD2
(add.rn.f32x2), an odd offset T scalar FADDs on the halves of the pairs (no register moves).
u16 : accumulators hold two 16-bit lanes (two consecutive samples) per 32-bit register.  gen_u16 keeps the window
in both phases (we[m] = samples 2m, 2m+1; wo[m] = samples 2m+1, 2m+2, one funnel shift per register); gen_u16p
(the default) keeps two accumulator rows per DM instead (even / odd offsets) and adds the window as loaded.

Run by build.py before nvcc; the output is committed so that the repository builds without Python.
"""
import os
import sys

F32_HEAD = os.environ.get('MDSM_GEN_F32_HEAD', 'rep')
U16_DISPATCH = os.environ.get('MDSM_GEN_U16_DISPATCH', 'shared')
U16_HEAD = os.environ.get('MDSM_GEN_U16_HEAD', 'shared')
DISPATCH = os.environ.get('MDSM_GEN_DISPATCH', 'tree')     # 'tree' (direct conditional branches) | 'brx' (indirect)


def tree_bits(e, j):
    """predicates b0..b3 <- bits of offset byte j of hi (issued early: they are ready long before the branches)"""
    for bit in range(4):
        e(f"and.b32 tm, hi, {1 << (8 * j + bit)}; setp.ne.u32 b{bit}, tm, 0;")


SKIP_LEAF = False        # set while generating a loop whose table entries may carry offset 15 = "this DM skips the row"


def tree_branch(e, j, noff):
    """branch to B{j}_{o}: at most 4 conditional direct branches, ~2 taken"""
    def leaf(k):
        if SKIP_LEAF and k == 15:
            return f"B{j}_15"
        return f"B{j}_{k}" if k < noff else f"B{j}_0"
    e(f"@b3 bra.uni X{j}_8; @b2 bra.uni X{j}_4; @b1 bra.uni X{j}_2; @b0 bra.uni {leaf(1)}; bra.uni {leaf(0)};")


def tree_stubs(e, j, noff):
    def leaf(k):
        if SKIP_LEAF and k == 15:
            return f"B{j}_15"
        return f"B{j}_{k}" if k < noff else f"B{j}_0"
    e(f"X{j}_2: @b0 bra.uni {leaf(3)}; bra.uni {leaf(2)};")
    e(f"X{j}_4: @b1 bra.uni X{j}_6; @b0 bra.uni {leaf(5)}; bra.uni {leaf(4)};")
    e(f"X{j}_6: @b0 bra.uni {leaf(7)}; bra.uni {leaf(6)};")
    e(f"X{j}_8: @b2 bra.uni X{j}_12; @b1 bra.uni X{j}_10; @b0 bra.uni {leaf(9)}; bra.uni {leaf(8)};")
    e(f"X{j}_10: @b0 bra.uni {leaf(11)}; bra.uni {leaf(10)};")
    e(f"X{j}_12: @b1 bra.uni X{j}_14; @b0 bra.uni {leaf(13)}; bra.uni {leaf(12)};")
    e(f"X{j}_14: @b0 bra.uni {leaf(15)}; bra.uni {leaf(14)};")


def nchunks(T, NOFF, per_chunk):
    """128-bit chunks holding T + NOFF - 1 samples"""
    return (T + NOFF - 1 + per_chunk - 1) // per_chunk


class Emit:
    def __init__(self):
        self.lines = []

    def __call__(self, s):
        self.lines.append(f'        "{s}\\n\\t"')


def gen_f32(D, T, NOFF):
    global SKIP_LEAF
    SKIP_LEAF = False
    try:
        return _gen_f32(D, T, NOFF)
    finally:
        SKIP_LEAF = False


def _gen_f32(D, T, NOFF):
    assert T % 4 == 0 and D <= 4
    A2 = T // 2
    NCH = nchunks(T, NOFF, 4)
    W2 = NCH * 2
    base_ch = T // 4
    assert NCH - base_ch <= 3
    nacc = D * A2
    SB, TAB = nacc, nacc + 1
    name = f"slab_f32_{D}_{T}_{NOFF}"
    e = Emit()
    e("{")
    e(f".reg .b64 w<{W2}>;")
    e(".reg .b32 lo, hi, p, tp, ix, tm;")
    e(".reg .pred q0, q1, q2, pl, b0, b1, b2, b3;")
    e(".reg .f32 a0, a1, x0, x1, y0, y1;")
    if DISPATCH == "brx":
        for j in range(D):
            e(f"ts{j}: .branchtargets " + ", ".join(f"B{j}_{k}" for k in range(NOFF)) + ";")

    def head():
        """decode the entry in (lo, hi), load the window, dispatch DM 0"""
        e("and.b32 p, lo, 0x3ffff; add.u32 p, p, %" + str(SB) + ";")
        for i in range(NCH - base_ch):
            e(f"and.b32 tm, lo, {1 << (28 + i)}; setp.ne.u32 q{i}, tm, 0;")
        e("setp.lt.s32 pl, lo, 0;")
        for i in range(NCH):
            pred = f"@q{i - base_ch} " if i >= base_ch else ""
            e(f"{pred}ld.shared.v2.b64 {{w{2 * i}, w{2 * i + 1}}}, [p+{16 * i}];")
        if DISPATCH == "brx":
            e("prmt.b32 ix, hi, 0, 0x4440; brx.idx ix, ts0;")
        else:
            tree_bits(e, 0)
            tree_branch(e, 0, NOFF)

    e(f"mov.u32 tp, %{TAB}; ld.shared.v2.b32 {{lo, hi}}, [tp];")
    e("HEAD:")
    head()
    for j in range(D):
        last = j == D - 1
        for k in list(range(NOFF)) + ([15] if SKIP_LEAF else []):
            m = k // 2
            e(f"B{j}_{k}:")
            if last:
                e("add.u32 tp, tp, 8; ld.shared.v2.b32 {lo, hi}, [tp];")      # next entry (garbage after the last one, unused)
            elif DISPATCH == "brx":
                e(f"prmt.b32 ix, hi, 0, 0x444{j + 1};")
            else:
                tree_bits(e, j + 1)
            body = ""
            for i in range(A2 if k < NOFF else 0):
                a = j * A2 + i
                if k % 2 == 0:
                    body += f"add.rn.f32x2 %{a}, %{a}, w{m + i}; "
                else:
                    body += (f"mov.b64 {{a0,a1}}, %{a}; mov.b64 {{x0,x1}}, w{m + i}; mov.b64 {{y0,y1}}, w{m + i + 1}; "
                             f"add.f32 a0, a0, x1; add.f32 a1, a1, y0; mov.b64 %{a}, {{a0,a1}}; ")
            e(body)
            if last:
                e("@pl bra.uni Bend;")
                if F32_HEAD == "shared":
                    e("bra.uni HEAD;")
                else:
                    head()
            elif DISPATCH == "brx":
                e(f"brx.idx ix, ts{j + 1};")
            else:
                tree_branch(e, j + 1, NOFF)
    if DISPATCH != "brx":
        for j in range(D):
            tree_stubs(e, j, NOFF)
    e("Bend:")
    e("}")
    s = [f"// f32x2 slab loop: D={D} DMs x T={T} samples, offsets < {NOFF}, {NCH} window chunks"]
    s.append(f"__device__ __forceinline__ void {name}(unsigned long long (&acc)[{D}][{A2}], unsigned sbase, unsigned tab)\n{{")
    s.append("    asm volatile(")
    s += e.lines
    s.append("        : " + ", ".join(f'"+l"(acc[{j}][{i}])' for j in range(D) for i in range(A2)))
    s.append('        : "r"(sbase), "r"(tab) : "memory");')
    s.append("}\n")
    s.append(f"template <> struct SlabF32<{D}, {T}, {NOFF}> {{ static constexpr int NCH = {NCH}; __device__ __forceinline__ static void run(unsigned long long (&a)[{D}][{A2}], unsigned sbase, unsigned tab) {{ {name}(a, sbase, tab); }} }};\n")
    return "\n".join(s)


def gen_f32p(D, T, NOFF):
    """fp32 loop of the pair pre-sum mode: a staged row is used by a SUBSET of the warp's DMs (bit 7 of a DM's offset
    byte = "skips this row").  The chain hops from one participating DM to the next: after its adds a block tests the
    skip bits of the DMs behind it (one predicated branch each) and enters the shared dispatcher DISP_j' of the first
    participant, or the loop tail when none is left.  One loop head (not copied), one dispatcher per DM slot; a block
    dispatches the NEXT slot itself when that slot uses the row (half of the time: one taken branch less)."""
    assert T % 4 == 0 and D <= 4
    A2 = T // 2
    NCH = nchunks(T, NOFF, 4)
    W2 = NCH * 2
    base_ch = T // 4
    assert NCH - base_ch <= 3
    nacc = D * A2
    SB, TAB = nacc, nacc + 1
    name = f"slab_f32p_{D}_{T}_{NOFF}"
    e = Emit()
    e("{")
    e(f".reg .b64 w<{W2}>;")
    e(".reg .b32 lo, hi, nlo, nhi, p, tp, tm;")
    e(".reg .pred q0, q1, q2, pl, b0, b1, b2, b3, s0, s1, s2, s3;")
    e(".reg .f32 a0, a1, x0, x1, y0, y1;")

    def skip_preds(first):
        for j in range(first, D):
            e(f"and.b32 tm, hi, {0x80 << (8 * j)}; setp.ne.u32 s{j}, tm, 0;")

    def hop(first):
        e(" ".join(f"@!s{j} bra.uni DISP{j};" for j in range(first, D)) + " bra.uni TAIL;")

    e(f"mov.u32 tp, %{TAB}; ld.shared.v2.b32 {{lo, hi}}, [tp];")
    e("bra.uni HEAD;")
    e("TAIL:")
    e("@pl bra.uni Bend;")
    e("add.u32 tp, tp, 8; mov.b32 lo, nlo; mov.b32 hi, nhi;")
    e("HEAD:")
    e("ld.shared.v2.b32 {nlo, nhi}, [tp+8];")                       # the entry after this one (unused after the last row)
    e("and.b32 p, lo, 0x3ffff; add.u32 p, p, %" + str(SB) + ";")
    for i in range(NCH - base_ch):
        e(f"and.b32 tm, lo, {1 << (28 + i)}; setp.ne.u32 q{i}, tm, 0;")
    e("setp.lt.s32 pl, lo, 0;")
    skip_preds(0)
    for i in range(NCH):
        pred = f"@q{i - base_ch} " if i >= base_ch else ""
        e(f"{pred}ld.shared.v2.b64 {{w{2 * i}, w{2 * i + 1}}}, [p+{16 * i}];")
    hop(0)
    for j in range(D):
        e(f"DISP{j}:")
        tree_bits(e, j)
        tree_branch(e, j, NOFF)
        tree_stubs(e, j, NOFF)
        if j + 1 < D:
            e(f"HOP{j}:")                      # slot j+1 skips the row: look further (rare enough to share the code)
            skip_preds(j + 2)
            hop(j + 2)
        for k in range(NOFF):
            m = k // 2
            e(f"B{j}_{k}:")
            if j + 1 < D:
                skip_preds_one = f"and.b32 tm, hi, {0x80 << (8 * (j + 1))}; setp.ne.u32 s{j + 1}, tm, 0;"
                e(skip_preds_one)
                tree_bits(e, j + 1)
            body = ""
            for i in range(A2):
                a = j * A2 + i
                if k % 2 == 0:
                    body += f"add.rn.f32x2 %{a}, %{a}, w{m + i}; "
                else:
                    body += (f"mov.b64 {{a0,a1}}, %{a}; mov.b64 {{x0,x1}}, w{m + i}; mov.b64 {{y0,y1}}, w{m + i + 1}; "
                             f"add.f32 a0, a0, x1; add.f32 a1, a1, y0; mov.b64 %{a}, {{a0,a1}}; ")
            e(body)
            if j + 1 < D:
                e(f"@s{j + 1} bra.uni HOP{j};")
                tree_branch(e, j + 1, NOFF)     # the next slot uses the row: dispatch it from here (one taken branch less)
            else:
                e("bra.uni TAIL;")
    e("Bend:")
    e("}")
    s = [f"// f32x2 slab loop, pair pre-sum mode: D={D} DMs x T={T} samples, offsets < {NOFF}, {NCH} window chunks"]
    s.append(f"__device__ __forceinline__ void {name}(unsigned long long (&acc)[{D}][{A2}], unsigned sbase, unsigned tab)\n{{")
    s.append("    asm volatile(")
    s += e.lines
    s.append("        : " + ", ".join(f'"+l"(acc[{j}][{i}])' for j in range(D) for i in range(A2)))
    s.append('        : "r"(sbase), "r"(tab) : "memory");')
    s.append("}\n")
    s.append(f"template <> struct SlabF32P<{D}, {T}, {NOFF}> {{ static constexpr int NCH = {NCH}; __device__ __forceinline__ static void run(unsigned long long (&a)[{D}][{A2}], unsigned sbase, unsigned tab) {{ {name}(a, sbase, tab); }} }};\n")
    return "\n".join(s)


def gen_u16(D, T, NOFF):
    """T samples = T/2 registers of two 16-bit lanes; window chunks of 8 samples (16 bytes of u16)."""
    assert T % 8 == 0 and D <= 4
    A = T // 2
    NCH = nchunks(T, NOFF, 8)
    WE = NCH * 4                      # registers of the even-phase window
    base_ch = T // 8
    assert NCH - base_ch <= 3
    nacc = D * A
    SB, TAB = nacc, nacc + 1
    name = f"slab_u16_{D}_{T}_{NOFF}"
    e = Emit()
    e("{")
    e(f".reg .b32 we<{WE}>, wo<{WE}>;")
    e(".reg .b32 lo, hi, p, tp, ix, tm;")
    e(".reg .pred q0, q1, q2, pl, b0, b1, b2, b3;")
    if DISPATCH == "brx":
        for j in range(D):
            e(f"ts{j}: .branchtargets " + ", ".join(f"B{j}_{k}" for k in range(NOFF)) + ";")

    def head():
        e("and.b32 p, lo, 0x3ffff; add.u32 p, p, %" + str(SB) + ";")
        for i in range(NCH - base_ch):
            e(f"and.b32 tm, lo, {1 << (28 + i)}; setp.ne.u32 q{i}, tm, 0;")
        e("setp.lt.s32 pl, lo, 0;")
        for i in range(NCH):
            pred = f"@q{i - base_ch} " if i >= base_ch else ""
            e(f"{pred}ld.shared.v4.b32 {{we{4 * i}, we{4 * i + 1}, we{4 * i + 2}, we{4 * i + 3}}}, [p+{16 * i}];")
        # odd phase: wo[m] = samples (2m+1, 2m+2) = funnel shift of (we[m], we[m+1]) right by 16 bits
        for m in range(WE - 1):
            e(f"shf.r.wrap.b32 wo{m}, we{m}, we{m + 1}, 16;")
        if DISPATCH == "brx":
            e("prmt.b32 ix, hi, 0, 0x4440; brx.idx ix, ts0;")
        elif U16_DISPATCH == "shared":
            e("bra.uni DISP0;")
        else:
            tree_bits(e, 0)
            tree_branch(e, 0, NOFF)

    e(f"mov.u32 tp, %{TAB}; ld.shared.v2.b32 {{lo, hi}}, [tp];")
    e("HEAD:")
    head()
    for j in range(D):
        last = j == D - 1
        for k in range(NOFF):
            m = k // 2
            src = "we" if k % 2 == 0 else "wo"
            e(f"B{j}_{k}:")
            if last:
                e("add.u32 tp, tp, 8; ld.shared.v2.b32 {lo, hi}, [tp];")
            elif DISPATCH == "brx":
                e(f"prmt.b32 ix, hi, 0, 0x444{j + 1};")
            elif U16_DISPATCH != "shared":
                tree_bits(e, j + 1)
            body = ""
            for i in range(A):
                a = j * A + i
                if i % 2 == 0:
                    body += f"add.u32 %{a}, %{a}, {src}{m + i}; "
                else:
                    body += f"mad.lo.u32 %{a}, {src}{m + i}, 1, %{a}; "
            e(body)
            if last:
                e("@pl bra.uni Bend;")
                if U16_HEAD == "shared":
                    e("bra.uni HEAD;")        # the u16 head (window loads + funnel shifts) is too long to copy 16 times
                else:
                    head()
            elif DISPATCH == "brx":
                e(f"brx.idx ix, ts{j + 1};")
            elif U16_DISPATCH == "shared":
                e(f"bra.uni DISP{j + 1};")
            else:
                tree_branch(e, j + 1, NOFF)
    if DISPATCH != "brx":
        for j in range(D):
            if U16_DISPATCH == "shared":      # one dispatcher per DM slot keeps the hot code inside the L1.5 I-cache
                e(f"DISP{j}:")
                tree_bits(e, j)
                tree_branch(e, j, NOFF)
            tree_stubs(e, j, NOFF)
    e("Bend:")
    e("}")
    s = [f"// u16x2 slab loop: D={D} DMs x T={T} samples, offsets < {NOFF}, {NCH} window chunks"]
    s.append(f"__device__ __forceinline__ void {name}(unsigned (&acc)[{D}][{A}], unsigned sbase, unsigned tab)\n{{")
    s.append("    asm volatile(")
    s += e.lines
    s.append("        : " + ", ".join(f'"+r"(acc[{j}][{i}])' for j in range(D) for i in range(A)))
    s.append('        : "r"(sbase), "r"(tab) : "memory");')
    s.append("}\n")
    s.append(f"template <> struct SlabU16<{D}, {T}, {NOFF}> {{ static constexpr int NCH = {NCH}; __device__ __forceinline__ static void run(unsigned (&a)[{D}][{A}], unsigned sbase, unsigned tab) {{ {name}(a, sbase, tab); }} }};\n")
    return "\n".join(s)


def gen_u16p(D, T, NOFF):
    """Two-phase u16x2 loop: no shifted window.  Every DM keeps TWO accumulator rows:
         E[i] = outputs (2i, 2i+1), i < T/2      fed by channels whose offset o = 2m is even:  E[i] += we[m+i]
         O[i] = outputs (2i-1, 2i), i <= T/2     fed by channels whose offset o = 2m+1 is odd: O[i] += we[m+i]
       (the outer halves of O[0] and O[T/2] belong to the neighbouring threads and are dropped); the epilogue adds
       the two rows.  Dispatch index = 8*(o & 1) + (o >> 1)."""
    assert T % 8 == 0 and D <= 4 and NOFF <= 16
    A = T // 2
    AW = 2 * A + 1
    NCH = nchunks(T, NOFF, 8)
    WE = NCH * 4
    base_ch = T // 8
    assert NCH - base_ch <= 3
    nacc = D * AW
    SB, TAB = nacc, nacc + 1
    name = f"slab_u16p_{D}_{T}_{NOFF}"
    e = Emit()
    e("{")
    e(f".reg .b32 we<{WE}>;")
    e(".reg .b32 lo, hi, p, tp, tm;")
    e(".reg .pred q0, q1, q2, pl, b0, b1, b2, b3;")

    def head():
        e("and.b32 p, lo, 0x3ffff; add.u32 p, p, %" + str(SB) + ";")
        for i in range(NCH - base_ch):
            e(f"and.b32 tm, lo, {1 << (28 + i)}; setp.ne.u32 q{i}, tm, 0;")
        e("setp.lt.s32 pl, lo, 0;")
        for i in range(NCH):
            pred = f"@q{i - base_ch} " if i >= base_ch else ""
            e(f"{pred}ld.shared.v4.b32 {{we{4 * i}, we{4 * i + 1}, we{4 * i + 2}, we{4 * i + 3}}}, [p+{16 * i}];")
        tree_bits(e, 0)
        tree_branch(e, 0, 16)

    e(f"mov.u32 tp, %{TAB}; ld.shared.v2.b32 {{lo, hi}}, [tp];")
    head()
    for j in range(D):
        last = j == D - 1
        for idx in range(16):
            odd, m = idx // 8, idx % 8
            e(f"B{j}_{idx}:")
            if 2 * m + odd >= NOFF:                 # unreachable index: keep the label, no code
                e("bra.uni Bend;")
                continue
            if last:
                e("add.u32 tp, tp, 8; ld.shared.v2.b32 {lo, hi}, [tp];")
            else:
                tree_bits(e, j + 1)
            body = ""
            n = A + 1 if odd else A
            for i in range(n):
                a = j * AW + (A + i if odd else i)
                if i % 2 == 0:
                    body += f"add.u32 %{a}, %{a}, we{m + i}; "
                else:
                    body += f"mad.lo.u32 %{a}, we{m + i}, 1, %{a}; "
            e(body)
            if last:
                e("@pl bra.uni Bend;")
                head()
            else:
                tree_branch(e, j + 1, 16)
    for j in range(D):
        tree_stubs(e, j, 16)
    e("Bend:")
    e("}")
    s = [f"// two-phase u16x2 slab loop: D={D} DMs x T={T} samples, offsets < {NOFF}, {NCH} window chunks"]
    s.append(f"__device__ __forceinline__ void {name}(unsigned (&acc)[{D}][{AW}], unsigned sbase, unsigned tab)\n{{")
    s.append("    asm volatile(")
    s += e.lines
    s.append("        : " + ", ".join(f'"+r"(acc[{j}][{i}])' for j in range(D) for i in range(AW)))
    s.append('        : "r"(sbase), "r"(tab) : "memory");')
    s.append("}\n")
    s.append(f"template <> struct SlabU16P<{D}, {T}, {NOFF}> {{ static constexpr int NCH = {NCH}; __device__ __forceinline__ static void run(unsigned (&a)[{D}][{AW}], unsigned sbase, unsigned tab) {{ {name}(a, sbase, tab); }} }};\n")
    return "\n".join(s)


def gen_u16pp(D, T, NOFF):
    """Two-phase u16x2 loop of the pair pre-sum mode: gen_u16p's add blocks (dispatch index = 8*(o & 1) + (o >> 1)) with
    gen_f32p's control flow (bit 7 of a DM's byte = the DM skips the row; hops, one dispatcher per DM slot, the next
    slot dispatched from inside the block when it uses the row)."""
    assert T % 8 == 0 and D <= 4 and NOFF <= 16
    A = T // 2
    AW = 2 * A + 1
    NCH = nchunks(T, NOFF, 8)
    WE = NCH * 4
    base_ch = T // 8
    assert NCH - base_ch <= 3
    nacc = D * AW
    SB, TAB = nacc, nacc + 1
    name = f"slab_u16pp_{D}_{T}_{NOFF}"
    e = Emit()
    e("{")
    e(f".reg .b32 we<{WE}>;")
    e(".reg .b32 lo, hi, nlo, nhi, p, tp, tm;")
    e(".reg .pred q0, q1, q2, pl, b0, b1, b2, b3, s0, s1, s2, s3;")

    def skip_preds(first):
        for j in range(first, D):
            e(f"and.b32 tm, hi, {0x80 << (8 * j)}; setp.ne.u32 s{j}, tm, 0;")

    def hop(first):
        e(" ".join(f"@!s{j} bra.uni DISP{j};" for j in range(first, D)) + " bra.uni TAIL;")

    e(f"mov.u32 tp, %{TAB}; ld.shared.v2.b32 {{lo, hi}}, [tp];")
    e("bra.uni HEAD;")
    e("TAIL:")
    e("@pl bra.uni Bend;")
    e("add.u32 tp, tp, 8; mov.b32 lo, nlo; mov.b32 hi, nhi;")
    e("HEAD:")
    e("ld.shared.v2.b32 {nlo, nhi}, [tp+8];")
    e("and.b32 p, lo, 0x3ffff; add.u32 p, p, %" + str(SB) + ";")
    for i in range(NCH - base_ch):
        e(f"and.b32 tm, lo, {1 << (28 + i)}; setp.ne.u32 q{i}, tm, 0;")
    e("setp.lt.s32 pl, lo, 0;")
    skip_preds(0)
    for i in range(NCH):
        pred = f"@q{i - base_ch} " if i >= base_ch else ""
        e(f"{pred}ld.shared.v4.b32 {{we{4 * i}, we{4 * i + 1}, we{4 * i + 2}, we{4 * i + 3}}}, [p+{16 * i}];")
    hop(0)
    for j in range(D):
        e(f"DISP{j}:")
        tree_bits(e, j)
        tree_branch(e, j, 16)
        tree_stubs(e, j, 16)
        if j + 1 < D:
            e(f"HOP{j}:")
            skip_preds(j + 2)
            hop(j + 2)
        for idx in range(16):
            odd, m = idx // 8, idx % 8
            e(f"B{j}_{idx}:")
            if 2 * m + odd >= NOFF:
                e("bra.uni Bend;")
                continue
            if j + 1 < D:
                e(f"and.b32 tm, hi, {0x80 << (8 * (j + 1))}; setp.ne.u32 s{j + 1}, tm, 0;")
                tree_bits(e, j + 1)
            body = ""
            n = A + 1 if odd else A
            for i in range(n):
                a = j * AW + (A + i if odd else i)
                if i % 2 == 0:
                    body += f"add.u32 %{a}, %{a}, we{m + i}; "
                else:
                    body += f"mad.lo.u32 %{a}, we{m + i}, 1, %{a}; "
            e(body)
            if j + 1 < D:
                e(f"@s{j + 1} bra.uni HOP{j};")
                tree_branch(e, j + 1, 16)
            else:
                e("bra.uni TAIL;")
    e("Bend:")
    e("}")
    s = [f"// two-phase u16x2 slab loop, pair pre-sum mode: D={D} DMs x T={T} samples, offsets < {NOFF}, {NCH} window chunks"]
    s.append(f"__device__ __forceinline__ void {name}(unsigned (&acc)[{D}][{AW}], unsigned sbase, unsigned tab)\n{{")
    s.append("    asm volatile(")
    s += e.lines
    s.append("        : " + ", ".join(f'"+r"(acc[{j}][{i}])' for j in range(D) for i in range(AW)))
    s.append('        : "r"(sbase), "r"(tab) : "memory");')
    s.append("}\n")
    s.append(f"template <> struct SlabU16PP<{D}, {T}, {NOFF}> {{ static constexpr int NCH = {NCH}; __device__ __forceinline__ static void run(unsigned (&a)[{D}][{AW}], unsigned sbase, unsigned tab) {{ {name}(a, sbase, tab); }} }};\n")
    return "\n".join(s)


# (D, T, NOFF) instances compiled into the library
F32_VARIANTS = [(4, 28, 12), (4, 20, 12), (2, 28, 12)]
U16_VARIANTS = [(4, 40, 16)]
U16P_VARIANTS = [(2, 40, 12), (3, 40, 14)]
F32P_VARIANTS = [(4, 28, 12), (4, 20, 12)]
U16PP_VARIANTS = [(2, 40, 12)]


def main(out):
    parts = ["// GENERATED by gen_chain.py -- do not edit.\n#pragma once\n"]
    parts.append("template <int D, int T, int NOFF> struct SlabF32;   // packed f32x2 slab loop\n")
    parts.append("template <int D, int T, int NOFF> struct SlabU16;   // packed u16x2 slab loop\n")
    parts.append("template <int D, int T, int NOFF> struct SlabU16P;  // two-phase packed u16x2 slab loop\n")
    parts.append("template <int D, int T, int NOFF> struct SlabF32P;  // packed f32x2 slab loop of the pair pre-sum mode\n")
    parts.append("template <int D, int T, int NOFF> struct SlabU16PP; // two-phase packed u16x2 slab loop of the pair pre-sum mode\n")
    for v in F32_VARIANTS:
        parts.append(gen_f32(*v))
    for v in U16_VARIANTS:
        parts.append(gen_u16(*v))
    for v in U16P_VARIANTS:
        parts.append(gen_u16p(*v))
    for v in F32P_VARIANTS:
        parts.append(gen_f32p(*v))
    for v in U16PP_VARIANTS:
        parts.append(gen_u16pp(*v))
    txt = "\n".join(parts)
    if os.path.exists(out) and open(out).read() == txt:
        return
    open(out, "w").write(txt)


if __name__ == "__main__":
    main(sys.argv[1] if len(sys.argv) > 1 else os.path.join(os.path.dirname(os.path.abspath(__file__)), "chain_gen.h"))
