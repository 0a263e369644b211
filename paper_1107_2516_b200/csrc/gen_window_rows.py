"""Writes window_rows.inc: the per-channel add block of the register-window kernel as inline PTX.

    python paper_1107_2516_b200/csrc/gen_window_rows.py

For every supported T (pairs per thread and row) it emits

    rows7(u64 (&acc)[8][T], const u64 (&w)[T + 1], unsigned m)

which adds, for the rows j = 1..7 of a thread, the window pairs w[i + o_j] (i = 0..T-1) to
acc[j][i] with o_j = bit (j-1) of m.  All seven predicates are computed first; every row has two
variants of T packed adds (add.rn.f32x2 -> FADD2) selected by `bra.uni`: written in PTX because
(a) a predicate feeding a branch right away costs ~13 cycles on sm_100a, so they must all be set
before the first row, and (b) the branches are warp-uniform by construction, which ptxas cannot
prove from C++ (profiles/r1c_microbench.md).
build.py regenerates the .inc when this file is newer.
"""
import os

# (rows per thread D, pairs per row T): 8 rows up to T = 11, 4 rows up to T = 21 (240 registers)
COMBOS = ((6, 15), (5, 17), (4, 15), (4, 21), (5, 11), (6, 9))


def rows7(T, D=8):
    """All D rows of a thread (the function keeps its 8-row name).  Row 0 adds w[i]; rows 1 .. D-1 are
    two chains of row blocks, A (offset 0) and B (offset 1); a block falls through to the next row's
    block of the same chain and only branches when the next row's bit differs, which halves the number
    of taken branches compared with one diamond per row.  Row 0 sits between the predicate setup and
    the first branch (it covers the predicate latency) and inside the same asm statement: as separate
    C++ adds ptxas computed some of them out of place and copied the result back (4 IMAD.MOV per
    channel on the FMA pipe)."""
    NJ = D - 1
    W = D * T             # first window operand
    M = D * T + T + 1     # mask operand
    L = ["{ .reg .pred p<%d>; .reg .b32 t;" % NJ]
    for r in range(NJ):
        L.append("and.b32 t, %%%d, %d; setp.ne.u32 p%d, t, 0;" % (M, 1 << r, r))

    def adds(row, o):
        return ["add.rn.f32x2 %%%d, %%%d, %%%d;" % (row * T + i, row * T + i, W + i + o) for i in range(T)]

    L += adds(0, 0)
    L.append("@p0 bra.uni B0_%=;")
    for r in range(NJ):
        L.append("A%d_%%=:" % r)
        L += adds(r + 1, 0)
        if r + 1 < NJ:
            L.append("@p%d bra.uni B%d_%%=;" % (r + 1, r + 1))
    L.append("bra.uni E_%=;")
    for r in range(NJ):
        L.append("B%d_%%=:" % r)
        L += adds(r + 1, 1)
        if r + 1 < NJ:
            L.append("@!p%d bra.uni A%d_%%=;" % (r + 1, r + 1))
    L.append("E_%=:")
    L.append("}")
    body = "\n".join('        "%s\\n"' % s for s in L)
    outs = ", ".join('"+l"(acc[%d][%d])' % (r, i) for r in range(D) for i in range(T))
    ins = ", ".join('"l"(w[%d])' % k for k in range(T + 1))
    return ("__device__ __forceinline__ void rows7(u64 (&acc)[%d][%d], const u64 (&w)[%d], unsigned m)\n"
            "{\n    asm volatile(\n%s\n        : %s\n        : %s, \"r\"(m));\n}\n" % (D, T, T + 1, body, outs, ins))


def chan_loop(T, D):
    """The whole per-channel loop of a stage as ONE asm statement of threaded code:

        chan_loop(acc, m, hw, sp, ch, slot_bytes)

    m = word of the current channel, hw = shared-memory address of the next channel's word, sp = this
    thread's window base in the current channel's slot, ch = channels left in the stage.  Per channel:
    next word (ld.shared), T + 1 window loads, row 0, then ONE indirect branch (brx.idx over the
    2^(D-1) offset patterns of rows 1 .. D-1) into a straight-line block that adds the other rows and
    then does the next channel's loads and row 0 ITSELF before branching on: a channel costs exactly one
    taken branch (the two-chain version of rows7 takes two on average; forcing all offsets to 0 in an
    experiment, i.e. one taken branch fewer per channel, made the kernel 13 % faster).  Measured: 1.3 % over
    the chains for 4 rows (8 variants of ~1.4 KB), nothing for 5, much slower for 6 rows (32 variants no
    longer sit in the instruction cache), and a compact form with a shared tail is slower than either.  Leaves when the stage is done (ch == 0) or when the next channel has a row shift
    (m & SHIFT != 0: the caller shifts, clears those bits and comes back)."""
    NP = 1 << (D - 1)
    NA = D * T
    M, HW, SP, CH, SB = NA, NA + 1, NA + 2, NA + 3, NA + 4
    L = ["{ .reg .b64 w<%d>; .reg .b32 mn, t, a, idx; .reg .pred pe, ps;" % (T + 1)]

    def adds(row, o):
        return ["add.rn.f32x2 %%%d, %%%d, w%d;" % (row * T + i, row * T + i, i + o) for i in range(T)]

    def top(tag):
        # loads and row 0 of the channel whose word is m; exits first if it needs a row shift
        X = ["and.b32 t, %%%d, %d; setp.ne.u32 ps, t, 0; @ps bra.uni DONE_%%=;" % (M, 0x7fe0)]
        X.append("ld.shared.u32 mn, [%%%d];" % HW)
        X.append("shr.u32 t, %%%d, 18; and.b32 t, t, 0x3ff8; add.u32 a, %%%d, t;" % (M, SP))
        X += ["ld.shared.b64 w%d, [a+%d];" % (k, 8 * k) for k in range(T + 1)]
        X.append("and.b32 idx, %%%d, %d;" % (M, NP - 1))
        X += adds(0, 0)
        X.append("brx.idx.uni idx, TS_%=;")
        return X

    L.append("TS_%=: .branchtargets " + ", ".join("V%d_%%=" % p for p in range(NP)) + ";")
    L.append("setp.eq.u32 pe, %%%d, 0; @pe bra.uni DONE_%%=;" % CH)
    L += top("entry")
    for p in range(NP):
        L.append("V%d_%%=:" % p)
        for r in range(1, D):
            L += adds(r, (p >> (r - 1)) & 1)
        L.append("mov.b32 %%%d, mn; add.u32 %%%d, %%%d, 4; add.u32 %%%d, %%%d, %%%d; sub.u32 %%%d, %%%d, 1;"
                 % (M, HW, HW, SP, SP, SB, CH, CH))
        L.append("setp.eq.u32 pe, %%%d, 0; @pe bra.uni DONE_%%=;" % CH)
        L += top("v%d" % p)
    L.append("DONE_%=:")
    L.append("}")
    body = "\n".join('        "%s\\n"' % x for x in L)
    outs = ", ".join('"+l"(acc[%d][%d])' % (r, i) for r in range(D) for i in range(T))
    return ("__device__ __forceinline__ void chan_loop(u64 (&acc)[%d][%d], unsigned& m, unsigned& hw, unsigned& sp, unsigned& ch, unsigned slot_bytes)\n"
            "{\n    asm volatile(\n%s\n        : %s, \"+r\"(m), \"+r\"(hw), \"+r\"(sp), \"+r\"(ch)\n        : \"r\"(slot_bytes)\n        : \"memory\");\n}\n"
            % (D, T, body, outs))


def shift_row(T):
    """a[i] = a[i-1] (i = T-1 .. 1), a[0] = carry, as exact adds of -0.0 on tied operands: with plain
    copies or untied outputs ptxas rotates the accumulator registers inside the hot loop."""
    L = []
    for i in range(T - 1, 0, -1):
        L.append("add.rn.f32x2 %%%d, %%%d, %%%d;" % (i, i - 1, T + 1))
    L.append("add.rn.f32x2 %%0, %%%d, %%%d;" % (T, T + 1))
    body = "\n".join('        "%s\\n"' % x for x in L)
    outs = ", ".join('"+l"(a[%d])' % i for i in range(T))
    return ("__device__ __forceinline__ void shift_row(u64 (&a)[%d], u64 carry)\n"
            "{\n    const u64 nz = 0x8000000080000000ull;\n    asm volatile(\n%s\n        : %s\n        : \"l\"(carry), \"l\"(nz));\n}\n"
            % (T, body, outs))


def main():
    here = os.path.dirname(os.path.abspath(__file__))
    out = ["// GENERATED by gen_window_rows.py -- do not edit.\n"]
    for D, T in COMBOS:
        out.append(rows7(T, D))
        if D == 4 or (D == 5 and T <= 11):  # 8 variants; 16 pay while their code stays small (5 x 11: 48.6 -> 44.4 ms); with 5 rows (16) it is no faster than the chains, with 6 (32) far slower (I-cache)
            out.append(chan_loop(T, D))
    for T in sorted({t for _, t in COMBOS}):
        out.append(shift_row(T))
    with open(os.path.join(here, "window_rows.inc"), "w") as f:
        f.write("\n".join(out))


if __name__ == "__main__":
    main()
