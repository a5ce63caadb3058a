#!/usr/bin/env python
"""Generates ``subband_rows.inc`` — the channel loop of one pipeline stage of the SUBBAND kernel
(subband.cu) as ONE inline-PTX statement of threaded code.  ``python gen_subband_rows.py [D K S G]``
after changing a tile constant; the generated file is committed so that the build needs nvcc only,
subband.cu static_asserts that its constants (plan.h) match the ones the file was generated for, and
tests/test_abi_cpu.py checks that the committed file is what this script emits.

Why PTX: a thread owns D DM rows x K consecutive samples (accumulators in registers) and
holds the union of its rows' input windows in registers; row j needs window words [o_j, o_j + K) with
o_j known only at run time (warp-uniform).  Registers cannot be indexed dynamically, so the adds of a
row need a code body with static operands, reached through a jump.  nvcc turns a C++ ``switch`` into
select chains (13 predicated moves per add), so the bodies and the jumps are written here.

Shape of the code (profiles/r2_subband.md has the measurements behind each choice):

  * joint dispatch: the rows are taken in groups of G; a group's offsets (o_a, o_b, ...) form a pattern
    id (o_a*(S+2) + o_b)..., 8 bits per group in the channel's record, which indexes a jump table
    (``brx.idx`` -> SASS LDC + BRX) with one body per possible tuple.  The window base is 2-word
    aligned (LDS.64), so the smallest offset is 0 or 1, and the sub-bands are cut so that the offsets
    of a thread's rows spread by <= S;
  * adds are ``add.rn.f32x2`` (SASS FADD2: two fp32 adds per lane and issue slot) on aligned register
    pairs for even offsets; odd offsets use two scalar ``add.rn.f32`` on the halves of the accumulator
    pair (same fp32-pipe time, one more issue slot, no moves, no shifted copy of the window);
  * threaded code: the body of the LAST group ends with the jump into the NEXT channel's first group,
    so a channel costs D/G indirect branches and nothing else — no loop branch, no reconvergence
    point (the round-1 loop spent a third of its samples at four branch targets per channel);
  * window prefetch inside the last group's bodies: its adds are ordered by window pair, and as soon
    as pair m has been read for the last time the next channel's pair m is loaded into the same
    registers (``@pm ld.shared.b64``), so the LDS latency hides under the adds and no second window
    is needed (168 registers, 3 warps per scheduler);
  * the jump table of the first group has one more entry, EXIT, taken after the stage's last channel.

Operands of the statement: %0.. acc[j][k2] (b64, "+l"), then rp0 (u32 shared address of the warp's
record of the stage's first channel; consecutive channels REC_STRIDE bytes apart), slot0 (u32 shared
address of the lane's window origin in the first channel's slot), slot_bytes, nch (channels in this
stage, >= 1).  A record is {lo: pattern ids, 8 bits per group, group 0 lowest; hi: window base in
8-byte pairs}.
"""
import itertools
import os
import sys


def generate(D, K, S, G, rec_stride):
    assert D % G == 0 and (S + 2) ** G <= 255        # 8 bits per group
    K2, OM = K // 2, S + 1
    NP = (K + OM + 1) // 2                            # 8-byte pairs a thread loads per channel
    NG = D // G
    assert K % 2 == 0 and K2 % 2 == 1, "K/2 must be odd: LDS.64 lanes K/2 pairs apart are then conflict-free"
    NA = D * K2
    RP0, SLOT0, SLOTB, NCH = ("%%%d" % (NA + i) for i in range(4))

    def acc(j, k):
        return "%%%d" % (j * K2 + k)

    tuples = list(itertools.product(range(S + 2), repeat=G))   # id order: first row most significant
    valid = [max(t) - min(t) <= S for t in tuples]
    EXIT = len(tuples)
    L = ["{", ".reg .f32 lf<%d>, hf<%d>, al<%d>, ah<%d>;" % (NP, NP, G * K2, G * K2), ".reg .b64 w<%d>;" % NP,
         ".reg .b32 t<%d>, rlo, rhi, nlo, nhi, cnt, sa, rp, sl;" % NG, ".reg .pred pm;"]
    for g in range(NG):
        tgt = [("B%d_%d" % (g, i)) if v else "DONE" for i, v in enumerate(valid)] + (["DONE"] if g == 0 else [])
        L.append("TP%d: .branchtargets %s;" % (g, ", ".join(tgt)))

    def ids(src):
        out = []
        for g in range(NG):
            out.append("and.b32 t0, %s, 255;" % src if g == 0 else "bfe.u32 t%d, %s, %d, 8;" % (g, src, 8 * g))
        return out

    # stage prologue: first channel's record and window, second channel's record
    L += ["mov.u32 rp, %s;" % RP0, "mov.u32 sl, %s;" % SLOT0, "mov.u32 cnt, %s;" % NCH,
          "ld.shared.v2.u32 {rlo, rhi}, [rp];", "shl.b32 sa, rhi, 3;", "add.u32 sa, sa, sl;"]
    for m in range(NP):
        L.append("ld.shared.b64 w%d, [sa+%d];" % (m, 8 * m))
    L += ["add.u32 rp, rp, %d;" % rec_stride, "add.u32 sl, sl, %s;" % SLOTB, "ld.shared.v2.u32 {nlo, nhi}, [rp];"]
    L += ids("rlo")
    L.append("brx.idx.uni t0, TP0;")

    def rows(g, t, prefetch):
        """adds of group g for offsets t, ordered by window pair; with `prefetch`, the next channel's
        pair m is loaded right after the last read of this channel's pair m"""
        out = []
        for m in range(NP):
            split = False
            for jj, o in enumerate(t):
                j, q = g * G + jj, o >> 1
                if o & 1:
                    k1, k0 = m - q, m - q - 1       # al[k1] += hf_m ; ah[k0] += lf_m
                    if (0 <= k1 < K2 or 0 <= k0 < K2) and not split:
                        out.append("mov.b64 {lf%d, hf%d}, w%d;" % (m, m, m))
                        split = True
                    if 0 <= k0 < K2:
                        out += ["add.rn.f32 ah%d, ah%d, lf%d;" % (jj * K2 + k0, jj * K2 + k0, m),
                                "mov.b64 %s, {al%d, ah%d};" % (acc(j, k0), jj * K2 + k0, jj * K2 + k0)]
                    if 0 <= k1 < K2:
                        out += ["mov.b64 {al%d, ah%d}, %s;" % (jj * K2 + k1, jj * K2 + k1, acc(j, k1)),
                                "add.rn.f32 al%d, al%d, hf%d;" % (jj * K2 + k1, jj * K2 + k1, m)]
                else:
                    k = m - q
                    if 0 <= k < K2:
                        out.append("add.rn.f32x2 %s, %s, w%d;" % (acc(j, k), acc(j, k), m))
            if prefetch:
                out.append("@pm ld.shared.b64 w%d, [sa+%d];" % (m, 8 * m))
        return out

    for g in range(NG):
        last = g == NG - 1
        for i, (t, v) in enumerate(zip(tuples, valid)):
            if not v:
                continue
            L.append("B%d_%d:" % (g, i))
            if not last:
                L += rows(g, t, False)
                L.append("brx.idx.uni t%d, TP%d;" % (g + 1, g + 1))
                continue
            # last group: is there a next channel in this stage? its window address; then the adds with
            # the prefetch; then its pattern ids, the record after it, and the jump into its first group
            L += ["add.u32 cnt, cnt, -1;", "setp.ne.u32 pm, cnt, 0;", "shl.b32 sa, nhi, 3;", "add.u32 sa, sa, sl;"]
            L += rows(g, t, True)
            L += ids("nlo")
            L += ["@!pm mov.u32 t0, %d;" % EXIT, "add.u32 rp, rp, %d;" % rec_stride, "add.u32 sl, sl, %s;" % SLOTB,
                  "ld.shared.v2.u32 {nlo, nhi}, [rp];", "brx.idx.uni t0, TP0;"]
    L += ["DONE:", "}"]
    text = "\n".join('    "%s\\n"' % x for x in L)
    outs = ", ".join('"+l"(acc[%d][%d])' % (j, k) for j in range(D) for k in range(K2))
    head = ("// GENERATED by gen_subband_rows.py %d %d %d %d %d - do not edit.\n"
            "// One pipeline stage of the SUBBAND kernel as threaded code: per channel %d LDS.64 and %d jump(s) on a pattern id\n"
            "// into %d bodies each; the last group's bodies prefetch the next channel's window and jump straight into it.\n"
            % (D, K, S, G, rec_stride, NP, NG, sum(valid)))
    params = ("#ifdef SB_ROWS_PARAMS\n"
              "static_assert(SB_D == %d && SB_K == %d && SB_S == %d && SB_G == %d && SB_REC_STRIDE == %d, \"regenerate subband_rows.inc (gen_subband_rows.py)\");\n"
              "#else\n" % (D, K, S, G, rec_stride))
    return head + params + ("asm volatile(\n%s\n    : %s\n    : \"r\"(rp0), \"r\"(slot0), \"r\"(slot_bytes), \"r\"(nch)\n    : \"memory\");\n#endif\n" % (text, outs))


def generate_i16(D, K, OMAX, rec_stride):
    """The same stage loop for u8 plans that sum PACKED 16-bit pairs on the integer pipes (``subband_rows_i16.inc``).

    A 32-bit word holds two consecutive samples (the earlier one in the low half), a thread owns D rows x K
    words = 2K samples, and a row's in-window offset o (in SAMPLES, 0..OMAX) splits into a word offset o >> 1
    and a half-word bit: even offsets are K ``add.u32`` on whole words, odd ones K funnel-shift + add pairs that
    ptxas fuses into one ``LEA.HI`` each (acc + ((x[k+1] << 16) | (x[k] >> 16))).  No lane ever carries
    into its neighbour because a pass sums at most 257 channels of values <= 255 (plan.h SB16_CHMAX).
    Word offsets cost nothing here (no 64-bit register pairing), so every ROW jumps on its own offset: D
    jumps per channel and (OMAX + 1) bodies per row, for twice the samples of the fp32 loop.
    Operands: %0.. acc[j][k2] (b64 = two words = four samples, "+l"), then rp0, slot0, slot_bytes, nch as
    above; a record is {lo: one offset per row, 8 bits each, row 0 lowest; hi: window base in 8-byte pairs}."""
    assert K % 2 == 0 and OMAX + 1 <= 255
    K2 = K // 2
    NP = ((OMAX >> 1) + K + 1 + 1) // 2               # 8-byte pairs a thread loads per channel
    NA = D * K2
    RP0, SLOT0, SLOTB, NCH = ("%%%d" % (NA + i) for i in range(4))
    EXIT = OMAX + 1
    L = ["{", ".reg .b32 a<%d>, x<%d>, f<%d>;" % (D * K, 2 * NP, K),
         ".reg .b32 t<%d>, rlo, rhi, nlo, nhi, cnt, sa, rp, sl;" % D, ".reg .pred pm;"]
    for g in range(D):
        tgt = ["B%d_%d" % (g, o) for o in range(OMAX + 1)] + (["DONE"] if g == 0 else [])
        L.append("TP%d: .branchtargets %s;" % (g, ", ".join(tgt)))
    for i in range(NA):
        L.append("mov.b64 {a%d, a%d}, %%%d;" % (2 * i, 2 * i + 1, i))

    def ids(src):
        return ["and.b32 t0, %s, 255;" % src if g == 0 else "bfe.u32 t%d, %s, %d, 8;" % (g, src, 8 * g) for g in range(D)]

    def load(m, pred):
        return "%sld.shared.v2.b32 {x%d, x%d}, [sa+%d];" % ("@pm " if pred else "", 2 * m, 2 * m + 1, 8 * m)

    L += ["mov.u32 rp, %s;" % RP0, "mov.u32 sl, %s;" % SLOT0, "mov.u32 cnt, %s;" % NCH,
          "ld.shared.v2.u32 {rlo, rhi}, [rp];", "shl.b32 sa, rhi, 3;", "add.u32 sa, sa, sl;"]
    L += [load(m, False) for m in range(NP)]
    L += ["add.u32 rp, rp, %d;" % rec_stride, "add.u32 sl, sl, %s;" % SLOTB, "ld.shared.v2.u32 {nlo, nhi}, [rp];"]
    L += ids("rlo")
    L.append("brx.idx.uni t0, TP0;")

    def rows(j, o, prefetch):
        ow, ob = o >> 1, o & 1
        out = []
        if prefetch:                                    # pairs this row never reaches from below
            out += [load(m, True) for m in range(NP) if 2 * m + 1 < ow]
        for k in range(K):
            acc = "a%d" % (j * K + k)
            if ob:
                out += ["shf.r.wrap.b32 f%d, x%d, x%d, 16;" % (k, k + ow, k + ow + 1), "add.u32 %s, %s, f%d;" % (acc, acc, k)]
            else:
                out.append("add.u32 %s, %s, x%d;" % (acc, acc, k + ow))
            if prefetch and (k + ow) & 1:
                out.append(load((k + ow) >> 1, True))  # both words of this pair have been read for the last time
        if prefetch:                                    # the pair the last add straddles or stops in, and those above
            done = {m for m in range(NP) if 2 * m + 1 < ow} | {(k + ow) >> 1 for k in range(K) if (k + ow) & 1}
            out += [load(m, True) for m in range(NP) if m not in done]
        return out

    for g in range(D):
        last = g == D - 1
        for o in range(OMAX + 1):
            L.append("B%d_%d:" % (g, o))
            if not last:
                L += rows(g, o, False)
                L.append("brx.idx.uni t%d, TP%d;" % (g + 1, g + 1))
                continue
            L += ["add.u32 cnt, cnt, -1;", "setp.ne.u32 pm, cnt, 0;", "shl.b32 sa, nhi, 3;", "add.u32 sa, sa, sl;"]
            L += rows(g, o, True)
            L += ids("nlo")
            L += ["@!pm mov.u32 t0, %d;" % EXIT, "add.u32 rp, rp, %d;" % rec_stride, "add.u32 sl, sl, %s;" % SLOTB,
                  "ld.shared.v2.u32 {nlo, nhi}, [rp];", "brx.idx.uni t0, TP0;"]
    L.append("DONE:")
    for i in range(NA):
        L.append("mov.b64 %%%d, {a%d, a%d};" % (i, 2 * i, 2 * i + 1))
    L.append("}")
    text = "\n".join('    "%s\\n"' % x for x in L)
    outs = ", ".join('"+l"(acc[%d][%d])' % (j, k) for j in range(D) for k in range(K2))
    head = ("// GENERATED by gen_subband_rows.py (generate_i16 %d %d %d %d) - do not edit.\n"
            "// One pipeline stage of the SUBBAND kernel for packed 16-bit sums: per channel %d LDS.64 and one jump per row on its\n"
            "// own offset into %d bodies; the last row's bodies prefetch the next channel's window and jump straight into it.\n"
            % (D, K, OMAX, rec_stride, NP, OMAX + 1))
    params = ("#ifdef SB_ROWS_PARAMS\n"
              "static_assert(SB_D == %d && SB_K == %d && SB16_OMAX == %d && SB_REC_STRIDE == %d && SB16_WPAIRS == %d, \"regenerate subband_rows_i16.inc (gen_subband_rows.py)\");\n"
              "#else\n" % (D, K, OMAX, rec_stride, NP))
    return head + params + ("asm volatile(\n%s\n    : %s\n    : \"r\"(rp0), \"r\"(slot0), \"r\"(slot_bytes), \"r\"(nch)\n    : \"memory\");\n#endif\n" % (text, outs))


DEFAULT = (4, 26, 5, 2, 96)
DEFAULT_I16 = (4, 26, int(os.environ.get('SB16_OMAX', '11')), 96)

if __name__ == "__main__":
    a = [int(x) for x in sys.argv[1:]]
    a = tuple(a) + DEFAULT[len(a):]
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "subband_rows.inc")
    with open(path, "w") as f:
        f.write(generate(*a))
    print(path, *a)
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "subband_rows_i16.inc")
    with open(path, "w") as f:
        f.write(generate_i16(a[0], a[1], DEFAULT_I16[2], a[4]))
    print(path, a[0], a[1], DEFAULT_I16[2], a[4])
