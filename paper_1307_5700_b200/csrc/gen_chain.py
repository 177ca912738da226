#!/usr/bin/env python
"""Generates chain_gen.h: the register-window accumulate chains of the tiled dedispersion kernels.

    chain_f32<D,T,NOFF>(acc2[D][T/2], w2[(T+NOFF-1+3)/4*2], o[D]):
        for j < D:  acc[j][i] += w[o[j] + i],  i < T        (o[j] warp-uniform, 0 <= o[j] < NOFF)

Registers cannot be indexed dynamically, so every (j, offset) pair owns a straight-line block of
adds.  The blocks are THREADED: block (j, o[j]) ends with the indirect branch (PTX brx.idx -> SASS
LDC jump-table read + BRX) into block (j+1, o[j+1]), so one channel costs D indirect branches and no
branch back, and the jump-table read of the next block is issued while the current block's adds run.
Accumulators and window are packed f32x2 register pairs: an even offset is T/2 FADD2
(add.rn.f32x2), an odd offset T scalar FADDs on the halves of the pairs (no register moves).

chain_u16<D,T,NOFF> is the integer form: accumulators and window hold two 16-bit lanes per 32-bit
register (two consecutive samples); an even offset adds the aligned window registers, an odd offset
the funnel-shifted ones (wo[m] = (w[m] >> 16) | (w[m+1] << 16), built once per channel by the caller).

A C++ `switch` does not work here: nvcc either merges the cases into one add block fed by register
moves or emits a compare tree.  Run by build.py before nvcc; the output is committed so that the
repository builds without Python.
"""
import os
import sys


def wregs(T, NOFF):
    """window length in 32-bit words: T + NOFF - 1 rounded up to whole 128-bit chunks"""
    return (T + NOFF - 1 + 3) // 4 * 4


def gen_f32(D, T, NOFF):
    assert T % 2 == 0
    A2 = T // 2
    W2 = wregs(T, NOFF) // 2
    nacc = D * A2
    name = f"chain_f32_{D}_{T}_{NOFF}"
    s = [f"// f32x2 chain: D={D} DMs x T={T} samples, offsets < {NOFF}"]
    s.append(f"__device__ __forceinline__ void {name}(unsigned long long (&acc)[{D}][{A2}], const unsigned long long (&w)[{W2}], unsigned lo, unsigned hi)\n{{")
    s.append('    asm volatile("{\\n\\t"')
    s.append('        ".reg .f32 a0, a1, x0, x1, y0, y1;\\n\\t"')
    s.append('        ".reg .b32 ix;\\n\\t"')
    for j in range(D):
        s.append(f'        "ts{j}: .branchtargets ' + ", ".join(f"B{j}_{k}" for k in range(NOFF)) + ';\\n\\t"')
    LO, HI = nacc + W2, nacc + W2 + 1

    def disp(j):
        # offset of DM j: byte 3 of lo (j = 0), byte j-1 of hi (j >= 1)
        src, byte = (LO, 3) if j == 0 else (HI, j - 1)
        return f"prmt.b32 ix, %{src}, 0, 0x444{byte}; brx.idx ix, ts{j};"

    s.append(f'        "{disp(0)}\\n\\t"')
    for j in range(D):
        for k in range(NOFF):
            m = k // 2
            body = ""
            for i in range(A2):
                a = j * A2 + i
                if k % 2 == 0:
                    body += f"add.rn.f32x2 %{a}, %{a}, %{nacc + m + i}; "
                else:
                    body += (f"mov.b64 {{a0,a1}}, %{a}; mov.b64 {{x0,x1}}, %{nacc + m + i}; mov.b64 {{y0,y1}}, %{nacc + m + i + 1}; "
                             f"add.f32 a0, a0, x1; add.f32 a1, a1, y0; mov.b64 %{a}, {{a0,a1}}; ")
            tail = disp(j + 1) if j + 1 < D else "bra.uni Bend;"
            s.append(f'        "B{j}_{k}: {body}{tail}\\n\\t"')
    s.append('        "Bend:\\n\\t"')
    s.append('        "}"')
    s.append("        : " + ", ".join(f'"+l"(acc[{j}][{i}])' for j in range(D) for i in range(A2)))
    s.append("        : " + ", ".join(f'"l"(w[{i}])' for i in range(W2)) + ', "r"(lo), "r"(hi));')
    s.append("}\n")
    s.append(f"template <> struct ChainF32<{D}, {T}, {NOFF}> {{ static constexpr int W2 = {W2}; __device__ __forceinline__ static void run(unsigned long long (&a)[{D}][{A2}], const unsigned long long (&w)[{W2}], unsigned lo, unsigned hi) {{ {name}(a, w, lo, hi); }} }};\n")
    return "\n".join(s)


def gen_u16(D, T, NOFF):
    """T samples = T/2 registers of two 16-bit lanes.  we[m] = samples (2m, 2m+1); wo[m] = samples (2m+1, 2m+2)."""
    assert T % 2 == 0
    A = T // 2
    WE = wregs(T, NOFF) // 2
    WO = WE - 1
    nacc = D * A
    name = f"chain_u16_{D}_{T}_{NOFF}"
    s = [f"// u16x2 chain: D={D} DMs x T={T} samples, offsets < {NOFF}"]
    s.append(f"__device__ __forceinline__ void {name}(unsigned (&acc)[{D}][{A}], const unsigned (&we)[{WE}], const unsigned (&wo)[{WO}], const unsigned (&o)[{D}])\n{{")
    s.append('    asm volatile("{\\n\\t"')
    for j in range(D):
        s.append(f'        "ts{j}: .branchtargets ' + ", ".join(f"B{j}_{k}" for k in range(NOFF)) + ';\\n\\t"')
    s.append(f'        "brx.idx %{nacc + WE + WO}, ts0;\\n\\t"')
    for j in range(D):
        for k in range(NOFF):
            m = k // 2
            base = nacc + m if k % 2 == 0 else nacc + WE + m
            body = "".join(f"add.u32 %{j * A + i}, %{j * A + i}, %{base + i}; " for i in range(A))
            tail = f"brx.idx %{nacc + WE + WO + j + 1}, ts{j + 1};" if j + 1 < D else "bra.uni Bend;"
            s.append(f'        "B{j}_{k}: {body}{tail}\\n\\t"')
    s.append('        "Bend:\\n\\t"')
    s.append('        "}"')
    s.append("        : " + ", ".join(f'"+r"(acc[{j}][{i}])' for j in range(D) for i in range(A)))
    s.append("        : " + ", ".join(f'"r"(we[{i}])' for i in range(WE)) + ", " + ", ".join(f'"r"(wo[{i}])' for i in range(WO)) + ", "
             + ", ".join(f'"r"(o[{j}])' for j in range(D)) + ");")
    s.append("}\n")
    s.append(f"template <> struct ChainU16<{D}, {T}, {NOFF}> {{ static constexpr int WE = {WE}; __device__ __forceinline__ static void run(unsigned (&a)[{D}][{A}], const unsigned (&we)[{WE}], const unsigned (&wo)[{WO}], const unsigned (&o)[{D}]) {{ {name}(a, we, wo, o); }} }};\n")
    return "\n".join(s)


# (D, T, NOFF) instances compiled into the library
F32_VARIANTS = [(4, 28, 12), (4, 20, 12), (5, 20, 16), (4, 28, 16)]
U16_VARIANTS = []


def main(out):
    parts = ["// GENERATED by gen_chain.py -- do not edit.\n#pragma once\n"]
    parts.append("template <int D, int T, int NOFF> struct ChainF32;   // packed f32x2 accumulate chain\n")
    parts.append("template <int D, int T, int NOFF> struct ChainU16;   // packed u16x2 accumulate chain\n")
    for v in F32_VARIANTS:
        parts.append(gen_f32(*v))
    for v in U16_VARIANTS:
        parts.append(gen_u16(*v))
    txt = "\n".join(parts)
    if os.path.exists(out) and open(out).read() == txt:
        return
    open(out, "w").write(txt)


if __name__ == "__main__":
    main(sys.argv[1] if len(sys.argv) > 1 else os.path.join(os.path.dirname(os.path.abspath(__file__)), "chain_gen.h"))
