#!/usr/bin/env python
"""Generates ``subband_rows.inc`` — the per-channel body of the SUBBAND kernel (subband.cu) as one
inline-PTX statement.  ``python gen_subband_rows.py joint [D K S G]`` (the committed joint-pattern body,
see generate_joint) or ``python gen_subband_rows.py D K OMAX [odd_mode [dispatch]]`` (the per-row body
described below, SB_JOINT_CFG=0) after changing a tile constant; the generated file is committed so that the build needs nvcc only, and subband.cu
static_asserts that its constants (plan.h) match the ones the file was generated for.

Why PTX: a thread owns SB_D DM rows x SB_K consecutive samples and holds the union of its rows'
input windows in registers; row j needs window words [o_j, o_j + SB_K) with o_j in 0..SB_OMAX known
only at run time (warp-uniform).  Registers cannot be indexed dynamically, so each row must reach one
of SB_OMAX+1 bodies with static register operands.  Measured on c3 (profiles/r1_subband.md):

  * a C++ ``switch`` is if-converted by nvcc into select chains (13 predicated moves per add): 9.5 %;
  * dispatch 1, "brx": threaded code, every body ends with the ``brx.idx`` of the next row (LDC from
    the jump table + BRX, ~88 cycles of warp latency per row): 15 %;
  * dispatch 0, "tree" (default of the per-row body): a binary tree of direct ``@q bra.uni`` on the four bits of o_j, the
    predicates set one body ahead; a taken direct branch costs ~12 cycles;
  * dispatch 2, "ttree": a private copy of the next row's tree in every body (no merge point, so no
    BSSY/BSYNC per row) — larger code, measured 1 % slower.

Adds are ``add.rn.f32x2`` (SASS FADD2: two fp32 adds per lane per issue slot).  FADD2 needs aligned
64-bit register pairs, which the window pairs as loaded provide for even o_j only.  Odd o_j:

  * odd_mode 1: a copy shifted by one word, built once per channel with ``or.b32 x, y, zero`` (``zero``
    is a run-time 0 so ptxas cannot turn the ORs into moves and sink them into every odd body);
    costs 2*NCHUNK*2 registers and ALU-pipe time;
  * odd_mode 0: plain moves; ptxas sinks 2 IMAD.MOV per FADD2 into the odd bodies — they run on the
    fp32 pipe and steal its cycles;
  * odd_mode 2 (default, also used by the joint body): two scalar ``add.rn.f32`` on the halves of the accumulator pair — the same
    fp32-pipe time as one FADD2, one more issue slot, no moves, no extra registers (this is what
    lets 3 warps per scheduler fit: 168 registers).

The per-row body tops out at 35 % of the add peak on c3 because every row pays a branch tree; the
joint body (generate_joint) dispatches once per group of rows and reaches 46 %.

The window's pad phase (where in the padded shared-memory layout the lane's first chunk falls) is
handled branch-free: chunk m sits at sa + 16*(m + m/P) + 16*[ar >= P - m%P].

Operands of the statement:  %0.. acc[j][k2] (b64, "+l"), then sa (u32 shared address of the lane's
first window chunk), ar (= a mod SB_K/4), obits (SB_D 4-bit o_j), zero.
"""
import os
import sys


def generate(D, K, OMAX, shifted_copy, dispatch="tree", head="arith"):
    K2 = K // 2
    P = K // 4                                  # chunks per lane = pad period (one pad chunk per P)
    NCHUNK = (K + OMAX + 3) // 4
    NW, NV, NO = 2 * NCHUNK, 2 * NCHUNK - 1, OMAX + 1
    assert D * 4 <= 32 and OMAX <= 15 and K % 4 == 0
    if P % 2 == 1:
        head = "linear"                         # odd chunk count per lane: the plain layout is conflict-free

    def acc(j, k):
        return "%%%d" % (j * K2 + k)

    SA, AR, OB, ZERO = ("%%%d" % (D * K2 + i) for i in range(4))
    L = ["{", ".reg .f32 al, ah, lf<%d>, hf<%d>;" % (NW, NW), ".reg .b32 t<%d>, tt;" % D, ".reg .pred q<4>;", ".reg .b64 w<%d>, v<%d>;" % (NW, NV),
         ".reg .b32 l<%d>, h<%d>, x<%d>, y<%d>;" % (NW, NW, NV, NV)]
    if head == "brx":
        L.append("TA: .branchtargets %s;" % ", ".join("LA%d" % r for r in range(P)))
    if dispatch == "brx":
        for j in range(D):
            L.append("T%d: .branchtargets %s;" % (j, ", ".join("R%d_%d" % (j, v) for v in range(NO))))

    def preds(j):
        # predicates q0..q3 = the four bits of o_j (tree dispatch); set one body ahead of their use
        out = []
        for b in range(4):
            if (1 << b) <= OMAX:
                out += ["and.b32 tt, %s, %d;" % (OB, 1 << (4 * j + b)), "setp.ne.u32 q%d, tt, 0;" % b]
        return out

    def goto_row(j):
        if j >= D:
            return ["bra.uni DONE;"]
        if dispatch == "brx":
            return ["brx.idx.uni t%d, T%d;" % (j, j)]
        if dispatch == "ttree":
            uid[0] += 1
            return jump_tree(j, 0, NO, 3, "c%d" % uid[0])   # private copy of row j's decision tree: no merge point
        return ["bra.uni TREE%d;" % j]

    uid = [0]

    def jump_tree(j, lo, hi, bit, tag):
        # decision tree whose leaves are jumps to the shared bodies R<j>_<o>
        if hi - lo == 1:
            return ["bra.uni R%d_%d;" % (j, lo)]
        mid = lo + (1 << bit)
        if mid >= hi:
            return jump_tree(j, lo, hi, bit - 1, tag)
        lab = "V%s_%d_%d_%d" % (tag, j, mid, bit)
        return (["@q%d bra.uni %s;" % (bit, lab)] + jump_tree(j, lo, mid, bit - 1, tag) + ["%s:" % lab] + jump_tree(j, mid, hi, bit - 1, tag))

    def body(j, o):
        out = ["R%d_%d:" % (j, o)]
        if dispatch in ("tree", "ttree") and j + 1 < D:
            out += preds(j + 1)
        for k in range(K2):
            if (o & 1) and shifted_copy == 2:
                # odd offset, no shifted copy: two scalar FADDs on the halves of the accumulator pair
                # (same fp32-pipe time as one FADD2, one more issue slot, no moves, no extra registers)
                i = (o >> 1) + k
                out += ["mov.b64 {al, ah}, %s;" % acc(j, k), "add.rn.f32 al, al, hf%d;" % i,
                        "add.rn.f32 ah, ah, lf%d;" % (i + 1), "mov.b64 %s, {al, ah};" % acc(j, k)]
            else:
                src = ("v%d" if o & 1 else "w%d") % ((o >> 1) + k)
                out.append("add.rn.f32x2 %s, %s, %s;" % (acc(j, k), acc(j, k), src))
        return out + goto_row(j + 1)

    def tree(j, lo, hi, bit):
        # binary decision tree over leaves [lo, hi) on bits bit..0 of o_j; the low half falls through
        if hi - lo == 1:
            return body(j, lo)
        mid = lo + (1 << bit)
        if mid >= hi:
            return tree(j, lo, hi, bit - 1)
        lab = "U%d_%d_%d" % (j, mid, bit)
        return (["@q%d bra.uni %s;" % (bit, lab)] + tree(j, lo, mid, bit - 1) + ["%s:" % lab] + tree(j, mid, hi, bit - 1))

    def after_loads():
        out = []
        if dispatch == "brx":
            for j in range(D):
                out.append("bfe.u32 t%d, %s, %d, 4;" % (j, OB, 4 * j))
        else:
            out += preds(0)
        for i in range(NW):
            out.append("mov.b64 {l%d, h%d}, w%d;" % (i, i, i))
        if shifted_copy == 2:
            for i in range(NW):
                out.append("mov.b64 {lf%d, hf%d}, w%d;" % (i, i, i))
            return out + goto_row(0)
        for i in range(NV):
            if shifted_copy:
                out.append("or.b32 x%d, h%d, %s;" % (i, i, ZERO))
                out.append("or.b32 y%d, l%d, %s;" % (i, i + 1, ZERO))
                out.append("mov.b64 v%d, {x%d, y%d};" % (i, i, i))
            else:
                out.append("mov.b64 v%d, {h%d, l%d};" % (i, i, i + 1))
        return out + goto_row(0)

    if head == "linear":
        for m in range(NCHUNK):
            L.append("ld.shared.v2.b64 {w%d, w%d}, [%s+%d];" % (2 * m, 2 * m + 1, SA, 16 * m))
        L += after_loads()
    elif head == "brx":
        # one jump on the pad phase ar into P copies of the loads with immediate offsets
        L.append("brx.idx.uni %s, TA;" % AR)
        for r in range(P):
            L.append("LA%d:" % r)
            for m in range(NCHUNK):
                off = 16 * (m + (r + m) // P)       # padded layout (subband.cu sb_phys)
                L.append("ld.shared.v2.b64 {w%d, w%d}, [%s+%d];" % (2 * m, 2 * m + 1, SA, off))
            L += after_loads()
    else:
        # branch-free: chunk m sits at sa + 16*(m + m/P) + 16*[ar >= P - m%P]  (one pad chunk per P)
        L.append(".reg .pred pa; .reg .b32 sx, b<%d>;" % P)
        L.append("mov.b32 b0, %s;" % SA)
        for rho in range(1, min(P, NCHUNK)):
            L += ["setp.ge.u32 pa, %s, %d;" % (AR, P - rho), "selp.b32 sx, 16, 0, pa;", "add.u32 b%d, %s, sx;" % (rho, SA)]
        for m in range(NCHUNK):
            L.append("ld.shared.v2.b64 {w%d, w%d}, [b%d+%d];" % (2 * m, 2 * m + 1, m % P, 16 * (m + m // P)))
        L += after_loads()
    for j in range(D):
        if dispatch in ("brx", "ttree"):
            for o in range(NO):
                L += body(j, o)
        else:
            L.append("TREE%d:" % j)
            L += tree(j, 0, NO, 3)
    L += ["DONE:", "}"]
    text = "\n".join('    "%s\\n"' % s for s in L)
    outs = ", ".join('"+l"(acc[%d][%d])' % (j, k) for j in range(D) for k in range(K2))
    ins = '"r"(sa), "r"(ar), "r"(obits), "r"(zero)'
    head = ("// GENERATED by gen_subband_rows.py %d %d %d %d - do not edit.\n"
            "// One channel of the SUBBAND kernel: window load (%d pad phases), shifted pairs, %d threaded row dispatches.\n"
            % (D, K, OMAX, shifted_copy, P, D))
    params = ("#ifdef SB_ROWS_PARAMS\n"
              "static_assert(SB_D == %d && SB_K == %d && SB_OMAX == %d, \"regenerate subband_rows.inc (gen_subband_rows.py)\");\n"
              "#else\n" % (D, K, OMAX))
    return head + params + "asm volatile(\n%s\n    : %s\n    : %s\n    : \"memory\");\n#endif\n" % (text, outs, ins)


def generate_joint(D, K, S, G=None):
    """SB_JOINT = 1: one dispatch per GROUP of G rows (default G = D: ONE per channel) on the joint
    offset pattern of the group's rows.

    The window is loaded as 8-byte pairs (LDS.64; with K/2 odd the plain layout is conflict-free), so
    its base is 2-word aligned and the smallest in-window offset is 0 or 1; the sub-bands are cut so
    that the offsets of a thread's rows spread by <= S.  A group's pattern id (o_a*(S+2) + o_b)*(S+2)...
    (8 bits per group in the record) indexes a jump table with one body per possible tuple holding the
    group's adds with static register operands; the body ends with the jump of the next group.  Only
    the few patterns that adjacent row groups and neighbouring channels actually produce are hot in the
    instruction cache (measured on c3: 16-18 of 122 for D = G = 3, S = 4), so the tables may be large."""
    import itertools
    G = D if G is None else G
    assert D % G == 0 and ((S + 2) ** G <= 256 or G == D)   # 8 bits per group; a single group owns the whole word
    K2, OM = K // 2, S + 1
    NP = (K + OM + 1) // 2
    NG = D // G
    assert K % 2 == 0 and K2 % 2 == 1, "K/2 must be odd: LDS.64 lanes K/2 pairs apart are then conflict-free"

    def acc(j, k):
        return "%%%d" % (j * K2 + k)

    SA, PID = "%%%d" % (D * K2), "%%%d" % (D * K2 + 1)
    L = ["{", ".reg .f32 al, ah, lf<%d>, hf<%d>;" % (NP, NP), ".reg .b64 w<%d>;" % NP, ".reg .b32 t<%d>;" % NG]
    tuples = list(itertools.product(range(S + 2), repeat=G))           # id order: first row most significant
    if NG == 1:   # the whole thread: min offset is 0 or 1 by construction
        valid = [min(t) <= 1 and max(t) - min(t) <= S for t in tuples]
    else:
        valid = [max(t) - min(t) <= S for t in tuples]
    for g in range(NG):
        L.append("TP%d: .branchtargets %s;" % (g, ", ".join(("B%d_%d" % (g, i)) if v else "DONE" for i, v in enumerate(valid))))
    for m in range(NP):
        L.append("ld.shared.b64 w%d, [%s+%d];" % (m, SA, 8 * m))
    for g in range(NG):
        L.append("bfe.u32 t%d, %s, %d, %d;" % (g, PID, 8 * g, 8 if NG > 1 else 16))
    for m in range(NP):
        L.append("mov.b64 {lf%d, hf%d}, w%d;" % (m, m, m))
    L.append("brx.idx.uni t0, TP0;")
    for g in range(NG):
        for i, (t, v) in enumerate(zip(tuples, valid)):
            if not v:
                continue
            L.append("B%d_%d:" % (g, i))
            for jj, o in enumerate(t):
                j = g * G + jj
                for k in range(K2):
                    m = (o >> 1) + k
                    if o & 1:   # odd offset: two scalar FADDs on the halves of the accumulator pair
                        L += ["mov.b64 {al, ah}, %s;" % acc(j, k), "add.rn.f32 al, al, hf%d;" % m,
                              "add.rn.f32 ah, ah, lf%d;" % (m + 1), "mov.b64 %s, {al, ah};" % acc(j, k)]
                    else:
                        L.append("add.rn.f32x2 %s, %s, w%d;" % (acc(j, k), acc(j, k), m))
            L.append("brx.idx.uni t%d, TP%d;" % (g + 1, g + 1) if g + 1 < NG else "bra.uni DONE;")
    L += ["DONE:", "}"]
    text = "\n".join('    "%s\\n"' % x for x in L)
    outs = ", ".join('"+l"(acc[%d][%d])' % (j, k) for j in range(D) for k in range(K2))
    head = ("// GENERATED by gen_subband_rows.py joint %d %d %d %d - do not edit.\n"
            "// One channel of the SUBBAND kernel, joint dispatch: %d LDS.64, %d jump(s) on a pattern id into %d bodies each.\n"
            % (D, K, S, G, NP, NG, sum(valid)))
    params = ("#ifdef SB_ROWS_PARAMS\n"
              "static_assert(SB_JOINT && SB_D == %d && SB_K == %d && SB_S == %d && SB_G == %d, \"regenerate subband_rows.inc (gen_subband_rows.py)\");\n"
              "#else\n" % (D, K, S, G))
    return head + params + "asm volatile(\n%s\n    : %s\n    : \"r\"(sa), \"r\"(obits)\n    : \"memory\");\n#endif\n" % (text, outs)


if __name__ == "__main__" and (len(sys.argv) < 2 or sys.argv[1] == "joint"):
    a = [int(x) for x in sys.argv[2:]]
    D, K, S = a[:3] if len(a) >= 3 else (4, 26, 5)
    G = a[3] if len(a) > 3 else (2 if len(a) < 3 else D)
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "subband_rows.inc")
    with open(path, "w") as f:
        f.write(generate_joint(D, K, S, G))
    print(path, "joint", D, K, S, G)
elif __name__ == "__main__":
    a = [int(x) for x in sys.argv[1:]]
    D, K, OMAX = a[:3] if len(a) >= 3 else (3, 28, 12)
    sc = a[3] if len(a) > 3 else 2
    disp = {0: "tree", 1: "brx", 2: "ttree"}[a[4] if len(a) > 4 else 0]
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "subband_rows.inc")
    with open(path, "w") as f:
        f.write(generate(D, K, OMAX, sc, disp))
    print(path, D, K, OMAX, sc)
