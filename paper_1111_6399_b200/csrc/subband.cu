// subband.cu — the SUBBAND kernel: exact sub-band re-skewed multi-pass brute-force de-dispersion
// with register-window reuse across adjacent DM trials.
//
// What it computes is still exactly out[d][t] = sum_c in[c][t + s(c,d)] (§2) with every
// (c,d) using its own rounded delay s(c,d) from the plan's table — no sub-band approximation.
//
// Why: one shared-memory word per add caps a kernel at 32 of the SM's 128 add lanes per clock
// (measured, profiles/r1_microbench.md). The paper's answer on Fermi — a thread keeps several time
// samples of one DM in registers and the block's (f,t) lines are reused from L1 —
// is kept, and extended: a thread owns SB_D adjacent DM trials x SB_K consecutive samples and loads
// the union of the SB_D windows ONCE into registers, so one loaded word feeds up to SB_D adds.
// That only pays when adjacent trials' delays differ by a few samples. The survey configs' DM plans
// are much coarser than the paper's (ndm = nchans), so the channels are split into sub-bands and
// each sub-band is processed in the skewed time coordinate u = t + s(c_ref, d): the residual delay
// r(c,d) = s(c,d) - s(c_ref,d) varies by <= SB_S samples across a thread's SB_D rows.
// One kernel launch per sub-band ("pass"); the first pass stores, later passes add into out.
//
// Per channel a thread: its record (prefetched one channel ahead), SB_WPAIRS LDS.64 of the window,
// then per group of SB_G rows ONE warp-uniform indirect branch on the group's joint offset pattern
// into a body with static register operands (registers cannot be indexed dynamically): SB_K/2 FADD2
// per row with an even offset, SB_K scalar FADD per row with an odd one. The channel loop of a whole
// pipeline stage is one generated inline-PTX statement of threaded code: the last group's bodies
// prefetch the next channel's window under their adds and jump straight into its first group (see
// gen_subband_rows.py for why and subband_rows.inc for the text). Around it: an SB_STAGES-deep ring
// filled by TMA bulk copies and handed over with mbarrier full/empty pairs (no CTA barrier in the
// loop), and a transposing epilogue that writes out with vector stores / red.global.add.v4.f32.
#include <algorithm>
#include <cstring>
#include <type_traits>

#include "plan.h"

namespace {

// Units of the window geometry. fp32 ring: a word is one sample. Packed 16-bit ring (u8 plans, SubbandGeom::i16):
// a word is two samples; everything below is in SAMPLES.
struct SbUnits {
    int aunit;      // samples per 8-byte window-base step
    int rb_align;   // the staged window starts at a multiple of this (one 16-byte chunk)
    int omax, spread;
    int ks;         // samples per thread and row
    int ws;         // samples in the window a thread loads (SB_WPAIRS pairs)
    int cs;         // samples per 16-byte chunk
    int chmax;      // channels per pass
    bool joint;     // record holds joint pattern ids per SB_G rows (fp32) / one offset per row (i16)
};
inline SbUnits sb_units(bool i16) {
    return i16 ? SbUnits{4, 8, SB16_OMAX, SB16_S, SB16_KS, 4 * SB16_WPAIRS, 8, SB16_CHMAX, false}
               : SbUnits{2, 4, SB_OMAX, SB_S, SB_K, 2 * SB_WPAIRS, 4, INT32_MAX, true};
}

// Residual-delay geometry of channels [cb, ce) against reference channel cr. Returns false if some
// group's in-window offsets would exceed SB_OMAX or a block's staged window exceeds SB_NCH_MAX.
// With `emit`, writes records/meta for those channels.
bool pass_geometry(dedisp_plan *p, int cb, int ce, int cr, bool emit, int b0, int b1) {
    const int ndm = p->ndm, ngroups = p->sb.ngroups, nblk = p->sb.nblk;
    const SbUnits U = sb_units(p->sb.i16);
    if (ce - cb > U.chmax) return false;
    const int32_t *sref = p->shifts.data() + (size_t)cr * ndm;
    const int gslots = nblk * SB_WARPS;
    std::vector<int> gmin(gslots), gmax(gslots);
    for (int c = cb; c < ce; ++c) {
        const int32_t *sc = p->shifts.data() + (size_t)c * ndm;
        for (int q = b0 * SB_WARPS; q < std::min(ngroups, b1 * SB_WARPS); ++q) {
            int mn = INT32_MAX, mx = INT32_MIN;
            for (int j = 0; j < SB_D; ++j) {
                const int d = std::min(q * SB_D + j, ndm - 1);
                const int r = sc[d] - sref[d];
                mn = std::min(mn, r);
                mx = std::max(mx, r);
            }
            gmin[q] = mn;
            gmax[q] = mx;
        }
        for (int q = std::max(ngroups, b0 * SB_WARPS); q < std::min(gslots, b1 * SB_WARPS); ++q) { gmin[q] = gmin[ngroups - 1]; gmax[q] = gmax[ngroups - 1]; }
        for (int b = b0; b < b1; ++b) {
            int bmin = INT32_MAX;
            for (int w = 0; w < SB_WARPS; ++w) bmin = std::min(bmin, gmin[b * SB_WARPS + w]);
            const int rbase = bmin & ~(U.rb_align - 1);  // toward -inf, two's complement
            // window base of a group inside the block's staged region in 8-byte pairs; what is left of
            // the residual delays are the in-window offsets
            const int AUNIT = U.aunit;
            int amax = 0;
            for (int w = 0; w < SB_WARPS; ++w) {
                const int q = b * SB_WARPS + w;
                const int a = (gmin[q] - rbase) / AUNIT;
                if (gmax[q] - rbase - AUNIT * a > U.omax) return false;
                if (gmax[q] - gmin[q] > U.spread) return false;
                amax = std::max(amax, a);
                if (emit) {
                    uint64_t rec = (uint64_t)a << 32;
                    const int qq = std::min(q, ngroups - 1);
                    uint32_t lo = 0;
                    for (int j = 0; j < SB_D; ++j) {
                        const int d = std::min(qq * SB_D + j, ndm - 1);
                        const int o = (sc[d] - sref[d]) - rbase - AUNIT * a;
                        if (!U.joint) { lo |= (uint32_t)o << (8 * j); continue; }   // one offset per row
                        // 8 bits per dispatch group: pattern id, the group's first row most significant
                        const int g = j / SB_G, sh = 8 * g;
                        const uint32_t id = ((lo >> sh) & 255u) * (SB_S + 2) + (uint32_t)o;
                        lo = (lo & ~(255u << sh)) | (id << sh);
                    }
                    p->sb.records[((size_t)(q / SB_WARPS) * p->nchans + c) * SB_WARPS + q % SB_WARPS] = rec | lo;
                }
            }
            // staged 16-byte chunks: the furthest lane of the furthest group must find its whole window
            const int nch = (AUNIT * amax + U.ks * 31 + U.ws + U.cs - 1) / U.cs;
            if (nch > SB_NCH_MAX || amax > 0xffff) return false;
            if (emit) {
                p->sb.meta[((size_t)b * p->nchans + c) * 2 + 0] = rbase;
                p->sb.meta[((size_t)b * p->nchans + c) * 2 + 1] = nch;
                p->sb.max_nch = std::max(p->sb.max_nch, nch);
            }
        }
    }
    return true;
}

// Reference channel for [cb, ce): the one whose delay at the largest DM is closest to the middle of
// the sub-band's delay range (delays are proportional to f^-2 - f_top^-2, so this halves |r|).
int pick_ref(const dedisp_plan *p, int cb, int ce) {
    const int ndm = p->ndm;
    auto sl = [&](int c) { return (long long)p->shifts[(size_t)c * ndm + ndm - 1]; };
    const long long mid2 = sl(cb) + sl(ce - 1);
    int best = cb;
    long long bestd = INT64_MAX;
    int lo = cb, hi = ce - 1;  // sl is non-decreasing in c: binary search for 2*sl(c) >= mid2
    while (lo < hi) {
        const int m = (lo + hi) / 2;
        if (2 * sl(m) >= mid2) hi = m; else lo = m + 1;
    }
    for (int c = std::max(cb, lo - 1); c <= std::min(ce - 1, lo + 1); ++c) {
        const long long dd = std::llabs(2 * sl(c) - mid2);
        if (dd < bestd) { bestd = dd; best = c; }
    }
    return best;
}

}  // namespace

// raw path: bytes per raw channel slot (window bytes + up to 15 lead bytes, rounded up to 16, + one
// spare chunk the realigning loads may touch)
static int sb_raw_slot_bytes(int slot_chunks, int esize, int cs) { return ((slot_chunks * cs * esize + 15 + 15) & ~15) + 16; }

// dynamic shared memory of the SUBBAND kernel for `cb` channels per stage (esize > 0: raw path)
static size_t sb_smem_bytes(int cb, int slot_chunks, int esize, bool i16) {
    size_t b = (size_t)SB_STAGES * cb * slot_chunks * 16 + (size_t)(SB_STAGES * cb + 1) * SB_REC_STRIDE + 16 * SB_STAGES + 16;
    b = (b + 15) / 16 * 16;
    b += (size_t)SB_WARPS * (i16 ? SB16_EP_WORDS : SB_EP_WORDS) * sizeof(float);
    if (esize > 0) b += (size_t)cb * sb_raw_slot_bytes(slot_chunks, esize, sb_units(i16).cs);
    return b;
}


static void subband_build_as(dedisp_plan *p, const bool i16) {
    p->sb = SubbandGeom();
    SubbandGeom &sb = p->sb;
    const int nchans = p->nchans, ndm = p->ndm;
    sb.i16 = i16;
    sb.tile_t = i16 ? SB16_T : SB_T;
    sb.ngroups = (ndm + SB_D - 1) / SB_D;
    sb.nblk = (sb.ngroups + SB_WARPS - 1) / SB_WARPS;
    const size_t gslots = (size_t)sb.nblk * SB_WARPS;
    if ((double)nchans * gslots * 8.0 > 4.0e9) return;  // record table would not fit sensibly
    if (p->dtype == DEDISP_U8 && (double)nchans * 255.0 >= 16777216.0) return;  // fp32 sums must stay exact
    // DM-block ranges: a plan whose DM step changes (c4: 0.1 / 0.25 / 0.5) would force the sub-band width
    // of its coarsest part on all rows; blocks are therefore grouped by their adjacent-row delay step at
    // the lowest channel (within a factor 1.5) and every range gets its own sub-band partition.
    std::vector<int> range_begin;
    {
        const int32_t *slast = p->shifts.data() + (size_t)(nchans - 1) * ndm;
        double lo = 0, hi = 0;
        for (int b = 0; b < sb.nblk; ++b) {
            const int d0 = b * SB_ROWS, d1 = std::min(ndm, d0 + SB_ROWS);
            double step = d1 - d0 > 1 ? (double)(slast[d1 - 1] - slast[d0]) / (d1 - d0 - 1) : 0.0;
            step = std::max(step, 1.0);
            if (b == 0 || std::max(hi, step) > 1.5 * std::min(lo, step)) { range_begin.push_back(b); lo = hi = step; }
            else { lo = std::min(lo, step); hi = std::max(hi, step); }
        }
        if (range_begin.size() > 8) range_begin.assign(1, 0);   // erratic DM list: one range
        range_begin.push_back(sb.nblk);
    }
    sb.nranges = (int)range_begin.size() - 1;
    std::vector<std::vector<SubbandPass>> cuts(sb.nranges);
    for (int r = 0; r < sb.nranges; ++r) {
        const int b0 = range_begin[r], b1 = range_begin[r + 1];
        // greedy from the top of the band: extend each sub-band as far as the geometry admits (exponential
        // then binary search)
        std::vector<SubbandPass> cut;
        int cb = 0;
        while (cb < nchans) {
            auto ok = [&](int ce) { return pass_geometry(p, cb, ce, pick_ref(p, cb, ce), false, b0, b1); };
            if (!ok(cb + 1)) { sb = SubbandGeom(); return; }  // a single channel against itself always has r = 0; defensive
            int good = cb + 1, step = 1;
            while (good < nchans) {
                const int trial = std::min(nchans, good + step);
                if (ok(trial)) { good = trial; step *= 2; } else break;
            }
            int bad = std::min(nchans, good + step);  // first known-bad (or nchans if all good)
            if (good < nchans) {
                int lo = good, hi = bad;  // ok(lo) true, ok(hi) false
                while (hi - lo > 1) {
                    const int m = (lo + hi) / 2;
                    if (ok(m)) lo = m; else hi = m;
                }
                good = lo;
            }
            if (p->time_major && good < nchans) {   // time-major input: sub-bands (and so stages) start at multiples of 16 channels
                good = cb + (good - cb) / 16 * 16;
                if (good == cb) { sb = SubbandGeom(); return; }
            }
            SubbandPass ps;
            ps.c_begin = cb;
            ps.c_end = good;
            ps.blk_begin = b0;
            ps.blk_end = b1;
            cut.push_back(ps);
            cb = good;
            if (cut.size() > 2048) { sb = SubbandGeom(); return; }  // hopelessly coarse plan: use TILED
        }
        // the greedy cut leaves whatever remains to the last sub-band; a pass of a few channels still costs a
        // whole sweep over out (c3: 8 channels, 1.0 ms), so share the channels of the last two evenly
        if (cut.size() >= 2) {
            SubbandPass &u = cut[cut.size() - 2], &v = cut.back();
            const int mid = p->time_major ? (u.c_begin + v.c_end) / 32 * 16 : (u.c_begin + v.c_end) / 2;
            if (v.c_end - v.c_begin < (u.c_end - u.c_begin) / 2 && mid > u.c_begin && mid <= u.c_end &&
                pass_geometry(p, mid, v.c_end, pick_ref(p, mid, v.c_end), false, b0, b1)) {
                u.c_end = mid;
                v.c_begin = mid;
            }
        }
        for (size_t i = 0; i < cut.size(); ++i) {
            cut[i].c_ref = pick_ref(p, cut[i].c_begin, cut[i].c_end);
            cut[i].first = i == 0;
        }
        cuts[r] = cut;
    }
    // launch k runs the k-th sub-band of EVERY DM range (they touch disjoint rows of out, so their order
    // within a launch is free): a plan with three ranges (c4) needs a third of the launches, each with
    // three times the tiles to balance over the SMs
    sb.launch_begin.clear();
    for (size_t k = 0;; ++k) {
        bool any = false;
        for (int r = 0; r < sb.nranges; ++r)
            if (k < cuts[r].size()) {
                if (!any) sb.launch_begin.push_back((int)sb.passes.size());
                any = true;
                sb.passes.push_back(cuts[r][k]);
            }
        if (!any) break;
    }
    sb.launch_begin.push_back((int)sb.passes.size());
    sb.records.assign((size_t)nchans * gslots, 0);
    sb.meta.assign((size_t)nchans * sb.nblk * 2, 0);
    sb.skew.assign(sb.passes.size() * (size_t)ndm, 0);
    for (size_t g = 0; g < sb.passes.size(); ++g) {
        SubbandPass &ps = sb.passes[g];
        if (!pass_geometry(p, ps.c_begin, ps.c_end, ps.c_ref, true, ps.blk_begin, ps.blk_end)) { sb = SubbandGeom(); return; }
        const int32_t *sref = p->shifts.data() + (size_t)ps.c_ref * ndm;
        std::memcpy(sb.skew.data() + g * (size_t)ndm, sref, (size_t)ndm * sizeof(int32_t));
        ps.max_skew = sref[std::min(ndm, ps.blk_end * SB_ROWS) - 1];
    }
    // the kernel's dynamic shared memory (ring + records + transpose buffers) must fit the 227 KB a CTA may opt into
    if (!subband_smem_fits(p)) { sb = SubbandGeom(); return; }
    // as many channels per stage as fit the 227 KB a CTA may opt into (fewer, longer stages: fewer hand-overs)
    sb.slot_chunks = sb.max_nch + 1;
    const int esize = dtype_esize(p->dtype);
    sb.raw_slot_bytes = sb_raw_slot_bytes(sb.slot_chunks, esize, sb_units(i16).cs);
    auto pick = [&](int es, int &cb_out, size_t &smem_out) {
        cb_out = SB_CB;
        for (int cb = SB_CB_MAX; cb > SB_CB; --cb)
            if (sb_smem_bytes(cb, sb.slot_chunks, es, i16) <= 227u * 1024u) { cb_out = cb; break; }
        smem_out = sb_smem_bytes(cb_out, sb.slot_chunks, es, i16);
    };
    pick(0, sb.cb, sb.smem);
    pick(esize, sb.cb_raw, sb.smem_raw);
    sb.ok = true;
}

void subband_build(dedisp_plan *p) {
    // u8 plans sum packed 16-bit pairs on the integer pipes; should that geometry not be admitted, the fp32 one is tried
    if (p->dtype == DEDISP_U8 && !(p->flags & DEDISP_PLAN_NO_PACKED)) {
        subband_build_as(p, true);
        if (p->sb.ok) return;
    }
    subband_build_as(p, false);
}

// Rebuild s(c,d) from the packed records (+ meta + skew) and compare with the table: the records
// are all the kernel sees, so 0 mismatches means the kernel's address arithmetic encodes exactly
// the plan's delays.
long long subband_verify_records(const dedisp_plan *p) {
    const SubbandGeom &sb = p->sb;
    if (!sb.ok) return -1;
    const int ndm = p->ndm;
    const SbUnits U = sb_units(sb.i16);
    long long bad = 0;
    std::vector<int> seen(p->nchans, 0);   // DM blocks that cover channel c: every channel exactly once per block
    for (size_t g = 0; g < sb.passes.size(); ++g) {
        const SubbandPass &ps = sb.passes[g];
        for (int c = ps.c_begin; c < ps.c_end; ++c) {
            seen[c] += ps.blk_end - ps.blk_begin;
            if (ps.c_end - ps.c_begin > U.chmax) ++bad;
            for (int d = ps.blk_begin * SB_ROWS; d < std::min(ndm, ps.blk_end * SB_ROWS); ++d) {
                const int q = d / SB_D, j = d % SB_D, b = q / SB_WARPS;
                const uint64_t rec = sb.records[((size_t)b * p->nchans + c) * SB_WARPS + q % SB_WARPS];
                const int a = (int)((rec >> 32) & 0xffff);
                int o;
                if (U.joint) {
                    uint32_t id = ((uint32_t)rec >> (8 * (j / SB_G))) & 255u;
                    for (int jj = SB_G - 1; jj > j % SB_G; --jj) id /= (SB_S + 2);
                    o = (int)(id % (SB_S + 2));
                } else {
                    o = (int)(((uint32_t)rec >> (8 * j)) & 255u);
                }
                const int rbase = sb.meta[((size_t)b * p->nchans + c) * 2];
                const int nch = sb.meta[((size_t)b * p->nchans + c) * 2 + 1];
                const long long s = (long long)sb.skew[g * (size_t)ndm + d] + rbase + U.aunit * a + o;
                const int need = (U.aunit * a + U.ks * 31 + U.ws + U.cs - 1) / U.cs;
                if (s != p->shifts[(size_t)c * ndm + d] || need > nch || (rbase & (U.rb_align - 1)) || o > U.omax) ++bad;
            }
        }
    }
    for (int c = 0; c < p->nchans; ++c) bad += seen[c] != sb.nblk;
    return bad;
}

// =====================================================================================
// device side
// =====================================================================================
#include <cuda_fp16.h>

namespace {

// CTA = SB_WARPS consumer warps (three warpgroups, 160 registers each after setmaxnreg) + one producer
// warpgroup (32 registers; its first warp issues every copy of the ring). Persistent: one CTA per SM
// walks the launch's tiles round-robin, the producer streams the stages of consecutive tiles through
// the ring back to back, and every consumer warp runs its own epilogue from a private transpose
// buffer, so neither the ring fill of a tile nor its epilogue leaves the fp32 pipe idle. The ring is
// only SB_STAGES = 2 deep on purpose: the consumer warps then never drift more than one stage apart,
// which keeps the bodies they run hot in the instruction cache for each other (measured on c3: 4 stages
// free-running 123.9 ms, 4 stages with a consumer barrier per stage 118.8, 2 stages free-running 111.1).
constexpr int SB_CONSUMERS = SB_WARPS * 32;
constexpr int SB_THREADS = SB_CONSUMERS + 128;
// registers per thread after setmaxnreg: the direct fp32 kernel's producer only issues copies (32 are
// plenty); the raw path's producer warps convert, and with 32 registers their loop spilled to local
// memory, which has no L1 to speak of next to 200+ KB of shared memory (c5: 83.0 ms -> 77.3 ms with 56)
template <bool RAW> struct SbRegs { static constexpr int consumer = RAW ? 152 : 160, producer = RAW ? 56 : 32; };
static_assert(SB_CONSUMERS * SbRegs<false>::consumer + 128 * SbRegs<false>::producer <= 65536, "register file");
static_assert(SB_CONSUMERS * SbRegs<true>::consumer + 128 * SbRegs<true>::producer <= 65536, "register file");
static_assert(SB_STAGES >= 2, "ring depth");
static_assert(SB_CB_MAX <= 32 && SB_CB <= SB_CB_MAX, "one producer lane per staged channel");
static_assert(SB_NCH_MAX % 32 == 0, "staging loop");

// Staged layout: a channel's window is plain and contiguous (ONE TMA bulk copy); lanes are SB_K words
// apart and SB_K/2 is odd, so LDS.64 is conflict-free (16 consecutive lanes hit 16 different bank pairs).
static_assert(SB_K % 2 == 0 && (SB_K / 2) % 2 == 1, "K/2 odd: LDS.64 conflict-free in the plain layout");
#define SB_ROWS_PARAMS
#include "subband_rows.inc"
#include "subband_rows_i16.inc"
#undef SB_ROWS_PARAMS

__device__ __forceinline__ void sb_cp_async16_zs(unsigned sa, const void *gmem, int src_bytes) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(sa), "l"(gmem), "r"(src_bytes));
}
__device__ __forceinline__ void sb_mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared.b64 [%0], %1;\n" ::"r"(bar), "r"(count));
}
// TMA bulk copy global -> shared (SASS UBLKCP); completion is counted in bytes on `bar`
__device__ __forceinline__ void sb_bulk_g2s(unsigned dst, const void *src, unsigned bytes, unsigned bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void sb_mbar_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.expect_tx.relaxed.cta.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void sb_mbar_arrive(unsigned bar) {
    asm volatile("{\n.reg .b64 st;\nmbarrier.arrive.shared.b64 st, [%0];\n}\n" ::"r"(bar) : "memory");
}
// arrive on `bar` once all cp.async issued so far by this thread have landed (pending count unchanged)
__device__ __forceinline__ void sb_mbar_arrive_cp_async(unsigned bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared.b64 [%0];\n" ::"r"(bar) : "memory");
}
#ifndef SB_SLEEP_NS
#define SB_SLEEP_NS 256
#endif
#define SB_STR2(x) #x
#define SB_STR(x) SB_STR2(x)
// producer side: the slot is usually still being read, so sleep instead of spinning on the issue slots
// of the consumer warps that share this scheduler
__device__ __forceinline__ void sb_mbar_wait_sleep(unsigned bar, unsigned parity) {
    asm volatile("{\n.reg .pred p;\nWAIT_%=:\nmbarrier.try_wait.parity.shared.b64 p, [%0], %1, %2;\n@p bra.uni DONE_%=;\nnanosleep.u32 " SB_STR(SB_SLEEP_NS) ";\nbra.uni WAIT_%=;\nDONE_%=:\n}\n"
                 ::"r"(bar), "r"(parity), "r"(100000u) : "memory");
}
__device__ __forceinline__ void sb_mbar_wait(unsigned bar, unsigned parity) {
    asm volatile("{\n.reg .pred p;\nWAIT_%=:\nmbarrier.try_wait.parity.shared.b64 p, [%0], %1;\n@p bra.uni DONE_%=;\nbra.uni WAIT_%=;\nDONE_%=:\n}\n" ::"r"(bar), "r"(parity) : "memory");
}

struct SbArgs {
    const void *in;           // direct path: fp32, 16-byte aligned, strides % 4 == 0; raw path: any dtype / alignment
    long long in_stride;      // elements
    long long in_total;       // readable elements per beam starting at `in`
    long long in_beam;        // elements between beams
    void *out;
    long long out_stride, out_beam;
    long long nsamp_out;
    const uint64_t *records;  // [nblk][nchans][SB_WARPS]
    const int2 *meta;         // [nblk][nchans] {window base r relative to u (multiple of 4), 16-byte chunks to stage}
    const int32_t *skew;      // [npasses][ndm]
    const SbPassDev *passes;  // [npasses]
    int pass_lo, pass_hi;     // this launch runs passes [pass_lo, pass_hi) of the table
    int blk_lo, blk_hi;       // ... restricted to DM blocks [blk_lo, blk_hi)
    int ndm, nchans, nbeams;
    int slot_chunks;          // 16-byte chunks per staged channel slot
    int raw_slot_bytes;       // raw path: bytes per raw channel slot
    int cb;                   // channels per pipeline stage (SB_CB .. SB_CB_MAX)
    int first;                // 1: the launch's passes store, 0: every pass adds into out, 2: per pass (first sub-band of its DM range),
                              // 3: per pass (last sub-band of its range: launches in reverse order)
    int out_vec4;             // out rows are 16-byte aligned (base, row stride, beam stride): vector epilogue
};

typedef unsigned long long sb_u64;     // one aligned register pair = two fp32 accumulators (FADD2 operand)

// The CTA's next non-empty tile. Tiles of a pass are numbered beam-major, then u-tile, then DM block
// (neighbouring CTAs work on neighbouring DM blocks of the same u-tile and share input windows in L2);
// the tiles of all passes of the launch form one list dealt round-robin to the CTAs. The producer and
// the consumers walk it with identical arithmetic.
struct SbTile {
    int p, w, rot;            // cursor: pass, next tile index of this CTA within it (-1: pass not opened), list offset mod grid
    int blk, beam, c_begin, c_end, first;
    long long U0;
    const int32_t *skew;
};

template <int TT>   // u-samples per tile
__device__ __forceinline__ bool sb_next_tile(const SbArgs &A, SbTile &t) {
    const int grid = (int)gridDim.x;
    for (;;) {
        if (t.p >= A.pass_hi) return false;
        const SbPassDev P = A.passes[t.p];
        const int b0 = max(A.blk_lo, P.blk_begin), nb = min(A.blk_hi, P.blk_end) - b0;
        const int ntu = (int)((A.nsamp_out + P.max_skew + TT - 1) / TT);
        const int ntiles = nb > 0 ? A.nbeams * ntu * nb : 0;
        if (t.w < 0) t.w = ((int)blockIdx.x + grid - t.rot) % grid;
        if (t.w >= ntiles) { t.rot = (t.rot + ntiles % grid) % grid; ++t.p; t.w = -1; continue; }
        const int w = t.w;
        t.w += grid;
        t.blk = b0 + w % nb;
        const int rest = w / nb;
        t.beam = rest / ntu;
        t.U0 = (long long)(rest % ntu) * TT;
        t.skew = A.skew + (size_t)t.p * A.ndm;
        const int d_first = t.blk * SB_ROWS, d_last = min(A.ndm, d_first + SB_ROWS) - 1;
        // rows of this block are valid for u in [skew(d), skew(d) + nsamp_out)
        if (t.U0 + TT <= (long long)__ldg(t.skew + d_first) || t.U0 >= (long long)__ldg(t.skew + d_last) + A.nsamp_out) continue;
        t.c_begin = P.c_begin;
        t.c_end = P.c_end;
        t.first = A.first == 3 ? P.pad0 : P.first;   // 3: the passes run last sub-band first, so a range's LAST sub-band stores
        return true;
    }
}

// four fp32 samples from a raw staged window (shared memory, element type TIN) at byte offset `off`
template <typename TIN>
__device__ __forceinline__ float4 sb_raw4(unsigned raw_u32, unsigned off) {
    const unsigned wa = raw_u32 + (off & ~3u), sh = (off & 3u) * 8u;
    auto lds = [](unsigned a) { unsigned v; asm volatile("ld.shared.b32 %0, [%1];\n" : "=r"(v) : "r"(a)); return v; };
    if constexpr (std::is_same<TIN, uint8_t>::value) {
        const unsigned v = __funnelshift_r(lds(wa), lds(wa + 4), sh);
        return make_float4((float)(v & 255u), (float)((v >> 8) & 255u), (float)((v >> 16) & 255u), (float)(v >> 24));
    } else if constexpr (std::is_same<TIN, __half>::value) {
        const unsigned w0 = lds(wa), w1 = lds(wa + 4), w2 = lds(wa + 8);
        const unsigned a = __funnelshift_r(w0, w1, sh), b = __funnelshift_r(w1, w2, sh);
        const float2 fa = __half22float2(*reinterpret_cast<const __half2 *>(&a)), fb = __half22float2(*reinterpret_cast<const __half2 *>(&b));
        return make_float4(fa.x, fa.y, fb.x, fb.y);
    } else {
        return make_float4(__uint_as_float(lds(wa)), __uint_as_float(lds(wa + 4)), __uint_as_float(lds(wa + 8)), __uint_as_float(lds(wa + 12)));
    }
}
// eight u8 samples of a raw staged window at byte offset `off` as four words of packed 16-bit pairs
// (earlier sample in the low half)
__device__ __forceinline__ uint4 sb_raw8_u16(unsigned raw_u32, unsigned off) {
    const unsigned wa = raw_u32 + (off & ~3u), sh = (off & 3u) * 8u;
    auto lds = [](unsigned a) { unsigned v; asm volatile("ld.shared.b32 %0, [%1];\n" : "=r"(v) : "r"(a)); return v; };
    const unsigned w0 = lds(wa), w1 = lds(wa + 4), w2 = lds(wa + 8);
    const unsigned a = __funnelshift_r(w0, w1, sh), b = __funnelshift_r(w1, w2, sh);
    return make_uint4(__byte_perm(a, 0, 0x4140), __byte_perm(a, 0, 0x4342), __byte_perm(b, 0, 0x4140), __byte_perm(b, 0, 0x4342));
}
template <typename TIN> __device__ __forceinline__ float sb_to_f32(TIN v) { return (float)v; }
template <> __device__ __forceinline__ float sb_to_f32<__half>(__half v) { return __half2float(v); }

// TIN = input element type. RAW = false: fp32 rows whose base and pitches are 16-byte aligned are copied
// by TMA straight into the ring. RAW = true (u8 / f16 input, or fp32 rows of any alignment): the
// windows are TMA-copied as raw bytes (from the 16-byte boundary below their first sample) into a raw
// buffer, and the four producer warps convert them to fp32 into the ring - no pre-pass over the input
// and no fp32 copy of it in HBM.
//
// MODE 0: direct, 1: raw, 2..5: TIME-MAJOR packed input with 8 / 4 / 2 / 1 bits per sample (SURVEY.md §8(f)
// rank 2: corner turn + unpack fused into the staging step; PAPER.md:26 names the stage in front of the
// dispersion search, PAPER.md:42 the channel-major view this kernel wants). Row t of the input holds all
// channels of time sample t, first channel in the least significant bits; the plan cuts its sub-bands
// at multiples of 16 channels and a stage is exactly 16 channels, so a stage reads 2*nbits contiguous
// bytes per time sample. The four producer warps walk the union of the stage's windows one time sample
// per lane, load those bytes straight from global memory, and scatter the 16 values as fp32 into the 16
// channel windows of the ring: the corner turn costs no extra pass over the input and no staging buffer.
template <typename TIN, int MODE>
__global__ void __launch_bounds__(SB_THREADS, 1) dedisp_subband_kernel(const SbArgs A) {
    constexpr bool I16 = MODE >= 6;   // u8 plan summed as packed 16-bit pairs: ring words hold two samples (6: raw, 7..10: time-major)
    constexpr bool RAW = MODE == 1 || MODE == 6;
    constexpr int TT = I16 ? SB16_T : SB_T;                  // u-samples per tile
    constexpr int CS = I16 ? 8 : 4;                          // samples per staged 16-byte chunk
    constexpr int EPW = I16 ? SB16_EP_WORDS : SB_EP_WORDS;   // words of a warp's transpose buffer
    static_assert(!I16 || std::is_same<TIN, uint8_t>::value, "packed sums are for u8 input");
    constexpr int TMB = MODE == 2 || MODE == 7 ? 8 : MODE == 3 || MODE == 8 ? 4 : MODE == 4 || MODE == 9 ? 2 : MODE == 5 || MODE == 10 ? 1 : 0;   // time-major: bits per sample
    constexpr bool CONV = RAW || TMB != 0;                                                   // producer warps write the ring
    extern __shared__ __align__(16) unsigned char sb_smem[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const unsigned slot_bytes = (unsigned)A.slot_chunks * 16;
    const int CB = A.cb;
    const unsigned stage_bytes = CB * slot_bytes;
    // [ring: STAGES x CB x slot][records: (STAGES x CB + 1) x SB_WARPS x 8][full, empty, raw_full, raw_empty barriers]
    // [transpose buffers][raw: CB x raw_slot]
    const unsigned sdata_base = (unsigned)__cvta_generic_to_shared(sb_smem);
    const unsigned srec_base = sdata_base + SB_STAGES * stage_bytes;
    const unsigned bar_full = srec_base + (SB_STAGES * CB + 1) * SB_REC_STRIDE;
    const unsigned bar_empty = bar_full + 8u * SB_STAGES;
    const unsigned bar_raw_full = bar_empty + 8u * SB_STAGES, bar_raw_empty = bar_raw_full + 8u;
    const unsigned ep_off = (bar_raw_empty + 8u - sdata_base + 15u) & ~15u;
    const unsigned raw_base = sdata_base + ep_off + SB_WARPS * EPW * 4;
    if (tid == 0) {
#pragma unroll
        for (int b = 0; b < SB_STAGES; ++b) { sb_mbar_init(bar_full + 8u * b, CONV ? 4 : 32); sb_mbar_init(bar_empty + 8u * b, SB_WARPS); }
        sb_mbar_init(bar_raw_full, 1);
        sb_mbar_init(bar_raw_empty, 4);
    }
    __syncthreads();
    SbTile t;
    t.p = A.pass_lo; t.w = -1; t.rot = 0;
    int it = 0;                                          // stages handed through the ring so far (all tiles)

    if (warp >= SB_WARPS) {
        // ---------------- producer warpgroup: its first warp fills the ring
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;\n" ::"n"(SbRegs<CONV>::producer));
        if constexpr (TMB != 0) {
            const int pw = warp - SB_WARPS;
            const unsigned char *inb = reinterpret_cast<const unsigned char *>(A.in);
            while (sb_next_tile<TT>(A, t)) {
                const int2 *meta = A.meta + (size_t)t.blk * A.nchans;
                for (int c0 = t.c_begin; c0 < t.c_end; c0 += CB, ++it) {   // CB == 16, c0 % 16 == 0 (plan built with DEDISP_PLAN_TIME_MAJOR)
                    const int buf = it % SB_STAGES, k = it / SB_STAGES;
                    const unsigned full = bar_full + 8u * buf;
                    const int n = min(CB, t.c_end - c0);
                    // lane j < n: window of channel c0 + j in time samples [e0, e0 + nw)
                    const int2 mt = lane < n ? __ldg(meta + c0 + lane) : make_int2(0, 0);
                    const long long e0 = t.U0 + mt.x;
                    const int nw = CS * mt.y;
                    long long t_lo = lane < n ? e0 : (1ll << 62), t_hi = lane < n ? e0 + nw : -(1ll << 62);
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) {
                        t_lo = min(t_lo, __shfl_xor_sync(0xffffffffu, t_lo, o));
                        t_hi = max(t_hi, __shfl_xor_sync(0xffffffffu, t_hi, o));
                    }
                    if (k > 0) sb_mbar_wait_sleep(bar_empty + 8u * buf, (unsigned)((k - 1) & 1));
                    if (pw == 0 && lane == 0) {   // the stage's records: n x SB_WARPS, contiguous
                        sb_mbar_expect_tx(full, (unsigned)n * SB_REC_STRIDE);
                        sb_bulk_g2s(srec_base + buf * CB * SB_REC_STRIDE, A.records + ((size_t)t.blk * A.nchans + c0) * SB_WARPS, (unsigned)n * SB_REC_STRIDE, full);
                    }
                    // lane j keeps channel j's slot address minus its window start, and its window as [lo, lo + nw)
                    // in samples relative to the union's first sample
                    const int lo = (int)(e0 - t_lo);
                    const unsigned sbase = sdata_base + buf * stage_bytes + lane * slot_bytes - (I16 ? 2u : 4u) * (unsigned)lo;
                    const size_t col = (size_t)c0 * TMB / 8;                  // byte of channel c0 in a row
                    constexpr int NW = TMB == 8 ? 4 : TMB == 4 ? 2 : 1;       // 32-bit words per row: 16 channels
                    constexpr int NB = TMB == 8 ? 2 : 4;                      // rows per lane in flight: all loads first, then the scatter
                    if constexpr (I16) {
                        // packed ring: a lane takes PAIRS of consecutive time samples (window starts are even: multiples
                        // of 8 samples), so one 32-bit store per channel covers two samples
                        constexpr int NP2 = NB / 2 > 0 ? NB / 2 : 1;          // sample pairs per lane in flight
                        for (long long tb = t_lo + 64 * NP2 * pw; tb < t_hi; tb += 256 * NP2) {
                            unsigned w[NP2][2][NW];
#pragma unroll
                            for (int r = 0; r < NP2; ++r)
#pragma unroll
                                for (int h = 0; h < 2; ++h) {
                                    const long long ts = tb + 64 * r + 2 * lane + h;
#pragma unroll
                                    for (int q = 0; q < NW; ++q) w[r][h][q] = 0u;
                                    if (ts >= 0 && ts < A.in_total && ts < t_hi) {
                                        const unsigned char *src = inb + (size_t)ts * A.in_stride + col;
                                        if constexpr (TMB == 8) { const uint4 v = __ldg(reinterpret_cast<const uint4 *>(src)); w[r][h][0] = v.x; w[r][h][1] = v.y; w[r][h][2] = v.z; w[r][h][3] = v.w; }
                                        else if constexpr (TMB == 4) { const uint2 v = __ldg(reinterpret_cast<const uint2 *>(src)); w[r][h][0] = v.x; w[r][h][1] = v.y; }
                                        else if constexpr (TMB == 2) w[r][h][0] = __ldg(reinterpret_cast<const unsigned *>(src));
                                        else w[r][h][0] = __ldg(reinterpret_cast<const unsigned short *>(src));
                                    }
                                }
                            const int idx0 = (int)(tb - t_lo) + 2 * lane;
#pragma unroll
                            for (int j = 0; j < 16; ++j) {
                                constexpr unsigned per = 32 / TMB;
                                const int loj = __shfl_sync(0xffffffffu, lo, j);
                                const int nj = __shfl_sync(0xffffffffu, nw, j);
                                const unsigned bj = __shfl_sync(0xffffffffu, sbase, j) + 2u * (unsigned)idx0;
#pragma unroll
                                for (int r = 0; r < NP2; ++r) {
                                    const unsigned x0 = (w[r][0][j / per] >> ((j % per) * TMB)) & ((1u << TMB) - 1u);
                                    const unsigned x1 = (w[r][1][j / per] >> ((j % per) * TMB)) & ((1u << TMB) - 1u);
                                    if ((unsigned)(idx0 + 64 * r - loj) < (unsigned)nj)
                                        asm volatile("st.shared.b32 [%0], %1;\n" ::"r"(bj + 128u * r), "r"(x0 | (x1 << 16)) : "memory");
                                }
                            }
                        }
                    } else
                    for (long long tb = t_lo + 32 * NB * pw; tb < t_hi; tb += 128 * NB) {   // 32 * NB time samples per warp and step
                        unsigned w[NB][NW];
#pragma unroll
                        for (int r = 0; r < NB; ++r) {
                            const long long ts = tb + 32 * r + lane;
#pragma unroll
                            for (int q = 0; q < NW; ++q) w[r][q] = 0u;
                            if (ts >= 0 && ts < A.in_total && ts < t_hi) {
                                const unsigned char *src = inb + (size_t)ts * A.in_stride + col;
                                if constexpr (TMB == 8) { const uint4 v = __ldg(reinterpret_cast<const uint4 *>(src)); w[r][0] = v.x; w[r][1] = v.y; w[r][2] = v.z; w[r][3] = v.w; }
                                else if constexpr (TMB == 4) { const uint2 v = __ldg(reinterpret_cast<const uint2 *>(src)); w[r][0] = v.x; w[r][1] = v.y; }
                                else if constexpr (TMB == 2) w[r][0] = __ldg(reinterpret_cast<const unsigned *>(src));
                                else w[r][0] = __ldg(reinterpret_cast<const unsigned short *>(src));
                            }
                        }
                        const int idx0 = (int)(tb - t_lo) + lane;
#pragma unroll
                        for (int j = 0; j < 16; ++j) {
                            constexpr unsigned per = 32 / TMB;                // samples per 32-bit word
                            const int loj = __shfl_sync(0xffffffffu, lo, j);
                            const int nj = __shfl_sync(0xffffffffu, nw, j);
                            const unsigned bj = __shfl_sync(0xffffffffu, sbase, j) + 4u * (unsigned)idx0;
#pragma unroll
                            for (int r = 0; r < NB; ++r) {
                                const unsigned x = (w[r][j / per] >> ((j % per) * TMB)) & ((1u << TMB) - 1u);
                                if ((unsigned)(idx0 + 32 * r - loj) < (unsigned)nj)
                                    asm volatile("st.shared.f32 [%0], %1;\n" ::"r"(bj + 128u * r), "f"((float)x) : "memory");
                            }
                        }
                    }
                    __syncwarp();
                    if (lane == 0) sb_mbar_arrive(full);
                }
            }
            return;
        }
        if constexpr (RAW) {
            const int pw = warp - SB_WARPS;
            constexpr long long ES = (long long)sizeof(TIN);
            const long long in_bytes = A.in_total * ES;
            while (sb_next_tile<TT>(A, t)) {
                const char *inb = reinterpret_cast<const char *>(A.in) + (size_t)t.beam * A.in_beam * ES;
                const int2 *meta = A.meta + (size_t)t.blk * A.nchans;
                for (int c0 = t.c_begin; c0 < t.c_end; c0 += CB, ++it) {
                    const int buf = it % SB_STAGES, k = it / SB_STAGES;
                    const unsigned full = bar_full + 8u * buf;
                    const int n = min(CB, t.c_end - c0);
                    // window of channel c: samples [e0, e0 + 4 nch); raw bytes from the 16-byte boundary at or below
                    // its first sample (lead bytes in front). A window whose raw copy would leave the beam's byte
                    // range is not copied at all: its converter reads global memory with bounds checks.
                    auto window = [&](int c, long long &g, unsigned &lead, unsigned &rb, int &nch) -> bool {
                        const int2 mt = __ldg(meta + c);
                        nch = mt.y;
                        g = ((long long)c * A.in_stride + t.U0 + mt.x) * ES;
                        lead = (unsigned)((reinterpret_cast<uintptr_t>(inb) + (unsigned long long)g) & 15u);
                        rb = (lead + (unsigned)CS * (unsigned)mt.y * (unsigned)ES + 15u) & ~15u;
                        return g - lead >= 0 && g - lead + rb <= in_bytes;
                    };
                    if (pw == 0) {   // copy warp: lane l copies the raw window of channel c0 + l with one TMA bulk copy
                        if (it > 0) sb_mbar_wait_sleep(bar_raw_empty, (unsigned)((it - 1) & 1));
                        if (lane < n) {
                            long long g; unsigned lead, rb; int nch;
                            if (window(c0 + lane, g, lead, rb, nch)) {
                                sb_mbar_expect_tx(bar_raw_full, rb);
                                sb_bulk_g2s(raw_base + lane * (unsigned)A.raw_slot_bytes, inb + (g - lead), rb, bar_raw_full);
                            }
                        }
                        __syncwarp();
                        if (lane == 0) sb_mbar_arrive(bar_raw_full);
                    }
                    if (k > 0) sb_mbar_wait_sleep(bar_empty + 8u * buf, (unsigned)((k - 1) & 1));
                    if (pw == 0 && lane == 0) {   // the stage's records: n x SB_WARPS, contiguous
                        sb_mbar_expect_tx(full, (unsigned)n * SB_REC_STRIDE);
                        sb_bulk_g2s(srec_base + buf * CB * SB_REC_STRIDE, A.records + ((size_t)t.blk * A.nchans + c0) * SB_WARPS, (unsigned)n * SB_REC_STRIDE, full);
                    }
                    sb_mbar_wait(bar_raw_full, (unsigned)(it & 1));
                    for (int cc = pw; cc < n; cc += 4) {   // this warp converts channels pw, pw + 4, ... of the stage
                        long long g; unsigned lead, rb; int nch;
                        const bool interior = window(c0 + cc, g, lead, rb, nch);
                        const unsigned dst = sdata_base + buf * stage_bytes + cc * slot_bytes;
                        if constexpr (I16) {
                            if (interior) {
                                const unsigned raw = raw_base + cc * (unsigned)A.raw_slot_bytes;
                                for (int i = lane; i < nch; i += 32) {
                                    const uint4 v = sb_raw8_u16(raw, lead + 8u * i);
                                    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};\n" ::"r"(dst + 16u * i), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
                                }
                            } else {
                                const uint8_t *src = reinterpret_cast<const uint8_t *>(inb);
                                for (int i = lane; i < nch; i += 32) {
                                    unsigned v[4];
#pragma unroll
                                    for (int q = 0; q < 4; ++q) {
                                        const long long e = g + 8 * i + 2 * q;
                                        const unsigned lo = e >= 0 && e < A.in_total ? src[e] : 0u, hi = e + 1 >= 0 && e + 1 < A.in_total ? src[e + 1] : 0u;
                                        v[q] = lo | (hi << 16);
                                    }
                                    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};\n" ::"r"(dst + 16u * i), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]) : "memory");
                                }
                            }
                        } else if (interior) {
                            const unsigned raw = raw_base + cc * (unsigned)A.raw_slot_bytes;
                            for (int i = lane; i < nch; i += 32) {
                                const float4 v = sb_raw4<TIN>(raw, lead + 4u * (unsigned)ES * i);
                                asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};\n" ::"r"(dst + 16u * i), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
                            }
                        } else {
                            const TIN *src = reinterpret_cast<const TIN *>(inb);
                            const long long e0 = g / ES;
                            for (int i = lane; i < nch; i += 32) {
                                float v[4];
#pragma unroll
                                for (int q = 0; q < 4; ++q) {
                                    const long long e = e0 + 4 * i + q;
                                    v[q] = e >= 0 && e < A.in_total ? sb_to_f32<TIN>(src[e]) : 0.f;
                                }
                                asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};\n" ::"r"(dst + 16u * i), "f"(v[0]), "f"(v[1]), "f"(v[2]), "f"(v[3]) : "memory");
                            }
                        }
                    }
                    __syncwarp();
                    if (lane == 0) { sb_mbar_arrive(full); sb_mbar_arrive(bar_raw_empty); }
                }
            }
            return;
        }
        if (warp != SB_WARPS) return;
        while (sb_next_tile<TT>(A, t)) {
            const float *in = reinterpret_cast<const float *>(A.in) + (size_t)t.beam * A.in_beam;
            const int2 *meta = A.meta + (size_t)t.blk * A.nchans;
            const uint64_t *recs = A.records + (size_t)t.blk * A.nchans * SB_WARPS;
            for (int c0 = t.c_begin; c0 < t.c_end; c0 += CB, ++it) {
                const int buf = it % SB_STAGES, k = it / SB_STAGES;
                const unsigned full = bar_full + 8u * buf;
                if (k > 0) sb_mbar_wait_sleep(bar_empty + 8u * buf, (unsigned)((k - 1) & 1));
                const int n = min(CB, t.c_end - c0);
                // lane l stages channel c0 + l: an interior window is one TMA bulk copy
                const bool mine = lane < n;
                const int2 mt = mine ? __ldg(meta + c0 + lane) : make_int2(0, 0);
                const long long e0 = (long long)(c0 + lane) * A.in_stride + t.U0 + mt.x;
                const bool interior = e0 >= 0 && e0 + 4ll * mt.y <= A.in_total;
                const unsigned dst = sdata_base + buf * stage_bytes + lane * slot_bytes;
                if (mine && interior) {
                    sb_mbar_expect_tx(full, 16u * (unsigned)mt.y);
                    sb_bulk_g2s(dst, in + e0, 16u * (unsigned)mt.y, full);
                }
                // windows that cross either end of the input allocation: bounds-checked zero-filling
                // 16-byte cp.async by the whole warp, one such channel at a time
                unsigned edge = __ballot_sync(0xffffffffu, mine && !interior);
                while (edge) {
                    const int cc = __ffs(edge) - 1;
                    edge &= edge - 1;
                    const long long e0c = __shfl_sync(0xffffffffu, e0, cc);
                    const int nchc = __shfl_sync(0xffffffffu, mt.y, cc);
                    const unsigned dstc = sdata_base + buf * stage_bytes + cc * slot_bytes;
                    for (int ch = lane; ch < nchc; ch += 32) {
                        const long long e = e0c + 4ll * ch;
                        long long valid = e < 0 ? 0 : (A.in_total - e) * 4;
                        valid = valid < 0 ? 0 : (valid > 16 ? 16 : valid);
                        sb_cp_async16_zs(dstc + 16u * ch, valid ? (const void *)(in + e) : (const void *)in, (int)valid);
                    }
                }
                if (lane == 0) {   // the stage's records: n x SB_WARPS, contiguous
                    sb_mbar_expect_tx(full, (unsigned)n * SB_REC_STRIDE);
                    sb_bulk_g2s(srec_base + buf * CB * SB_REC_STRIDE, recs + (size_t)c0 * SB_WARPS, (unsigned)n * SB_REC_STRIDE, full);
                }
                sb_mbar_arrive_cp_async(full);
            }
        }
        return;
    }

    // ---------------- consumer warps
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;\n" ::"n"(SbRegs<CONV>::consumer));
    const unsigned sdata_u32 = sdata_base + 4u * SB_K * lane;
    float *ep = reinterpret_cast<float *>(sb_smem + ep_off) + (size_t)warp * EPW;
    while (sb_next_tile<TT>(A, t)) {
        sb_u64 acc[SB_D][SB_K / 2];
#pragma unroll
        for (int j = 0; j < SB_D; ++j)
#pragma unroll
            for (int k = 0; k < SB_K / 2; ++k) acc[j][k] = 0ull;

        for (int c0 = t.c_begin; c0 < t.c_end; c0 += CB, ++it) {
            const int buf = it % SB_STAGES;
            sb_mbar_wait(bar_full + 8u * buf, (unsigned)((it / SB_STAGES) & 1));
            const int nch = min(CB, t.c_end - c0);
            // the stage's channels, threaded: records are warp-uniform {x = pattern ids, y = window base in pairs}
            const unsigned rp0 = srec_base + (buf * CB * SB_WARPS + warp) * 8u;
            const unsigned slot0 = sdata_u32 + buf * stage_bytes;
            if constexpr (I16) {
#include "subband_rows_i16.inc"
            } else {
#include "subband_rows.inc"
            }
            __syncwarp();
            if (lane == 0) sb_mbar_arrive(bar_empty + 8u * buf);
        }

        // Epilogue: a lane holds SB_K consecutive samples of each row, so direct stores would touch 32
        // sectors per instruction. Each warp transposes row by row through its own buffer and writes /
        // adds out[d][t] with lanes on consecutive 16-byte groups; no other warp is involved. The row is
        // parked SHIFTED by sh = skew(d) mod 4 words, so that the groups that are 16-byte aligned in out
        // are 16-byte aligned in the buffer too: one LDS.128 + one vector store / reduction per group.
        float *out = reinterpret_cast<float *>(A.out) + (size_t)t.beam * A.out_beam;
        const int d0 = t.blk * SB_ROWS + warp * SB_D;
        const int first = A.first >= 2 ? t.first : A.first;
        const unsigned ep_u32 = (unsigned)__cvta_generic_to_shared(ep);
#pragma unroll
        for (int j = 0; j < SB_D; ++j) {
            const int d = d0 + j;
            if (d >= A.ndm) break;
            const long long t0 = t.U0 - (long long)__ldg(t.skew + d);      // t of the tile's sample 0
            float *orow = out + (size_t)d * A.out_stride;
            const int sh = A.out_vec4 ? (int)(t0 & 3) : 0;                 // word 4g of the buffer <-> t = t0 - sh + 4g
            __syncwarp();
            const unsigned wbase = ep_u32 + 4u * (unsigned)((I16 ? SB16_KS : SB_K) * lane + sh);
            if constexpr (I16) {
                // a 64-bit accumulator = four samples as 16-bit integers; as fp32: 0x4B00hhhh is 2^23 + h exactly
#pragma unroll
                for (int k2 = 0; k2 < SB_K / 2; ++k2) {
                    const unsigned lo = (unsigned)acc[j][k2], hi = (unsigned)(acc[j][k2] >> 32);
                    const float f0 = __uint_as_float(__byte_perm(lo, 0x4B000000u, 0x7610)) - 8388608.f, f1 = __uint_as_float(__byte_perm(lo, 0x4B000000u, 0x7632)) - 8388608.f;
                    const float f2 = __uint_as_float(__byte_perm(hi, 0x4B000000u, 0x7610)) - 8388608.f, f3 = __uint_as_float(__byte_perm(hi, 0x4B000000u, 0x7632)) - 8388608.f;
                    if (!(sh & 1)) {
                        asm volatile("st.shared.v2.f32 [%0], {%1, %2};\n" ::"r"(wbase + 16u * k2), "f"(f0), "f"(f1) : "memory");
                        asm volatile("st.shared.v2.f32 [%0], {%1, %2};\n" ::"r"(wbase + 16u * k2 + 8u), "f"(f2), "f"(f3) : "memory");
                    } else {
                        asm volatile("st.shared.f32 [%0], %1;\n" ::"r"(wbase + 16u * k2), "f"(f0) : "memory");
                        asm volatile("st.shared.f32 [%0], %1;\n" ::"r"(wbase + 16u * k2 + 4u), "f"(f1) : "memory");
                        asm volatile("st.shared.f32 [%0], %1;\n" ::"r"(wbase + 16u * k2 + 8u), "f"(f2) : "memory");
                        asm volatile("st.shared.f32 [%0], %1;\n" ::"r"(wbase + 16u * k2 + 12u), "f"(f3) : "memory");
                    }
                }
            } else if (!(sh & 1)) {
#pragma unroll
                for (int k2 = 0; k2 < SB_K / 2; ++k2)
                    asm volatile("st.shared.b64 [%0], %1;\n" ::"r"(wbase + 8u * k2), "l"(acc[j][k2]) : "memory");
            } else {
#pragma unroll
                for (int k2 = 0; k2 < SB_K / 2; ++k2) {
                    asm volatile("st.shared.b32 [%0], %1;\n" ::"r"(wbase + 8u * k2), "r"((unsigned)acc[j][k2]) : "memory");
                    asm volatile("st.shared.b32 [%0], %1;\n" ::"r"(wbase + 8u * k2 + 4u), "r"((unsigned)(acc[j][k2] >> 32)) : "memory");
                }
            }
            __syncwarp();
            auto put = [&](int w) {                              // one buffer word, bounds-checked
                const int sidx = w - sh;
                const long long tt = t0 + sidx;
                if (sidx >= 0 && sidx < TT && tt >= 0 && tt < A.nsamp_out) {
                    if (first) orow[tt] = ep[w];
                    else asm volatile("red.global.add.f32 [%0], %1;\n" ::"l"(orow + tt), "f"(ep[w]) : "memory");
                }
            };
            if (A.out_vec4) {
                // Valid buffer words [w_lo, w_hi): inside the tile (w - sh in [0, TT)) and inside the row (t in
                // [0, nsamp_out)); warp-uniform, found once per row. The whole 16-byte groups [gf_lo, gf_hi) go out
                // as one LDS.128 + one plain vector store (first pass) or one fire-and-forget vector reduction
                // (SASS REDG.E.ADD.F32x4; the SM never waits for out) each, NB at a time so that the shared-memory
                // latencies overlap; the up to 3 + 3 words left over at the two ends go out one by one from lanes 0..7.
                const long long lo64 = max((long long)sh, (long long)sh - t0), hi64 = min((long long)(sh + TT), A.nsamp_out - t0 + sh);
                const int w_lo = (int)min(max(lo64, 0ll), (long long)(TT + 8)), w_hi = (int)min(max(hi64, 0ll), (long long)(TT + 8));
                if (w_hi > w_lo) {
                    const int gf_lo = (w_lo + 3) >> 2, gf_hi = w_hi >> 2;
                    const unsigned long long obase = (unsigned long long)orow + 4ull * (unsigned long long)(t0 - sh);   // buffer word w <-> address obase + 4 w
                    constexpr int NG = (TT + 3 + 3) / 4, NB = 4;
#pragma unroll
                    for (int b = 0; b < (NG + 32 * NB - 1) / (32 * NB); ++b) {
                        float4 v[NB];
#pragma unroll
                        for (int q = 0; q < NB; ++q) {
                            // unconditional load (a group index past the buffer is folded back into it): only valid groups are stored
                            const int g = lane + 32 * (NB * b + q);
                            asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];\n" : "=f"(v[q].x), "=f"(v[q].y), "=f"(v[q].z), "=f"(v[q].w) : "r"(ep_u32 + 16u * (g < NG ? g : lane)));
                        }
#pragma unroll
                        for (int q = 0; q < NB; ++q) {
                            const int g = lane + 32 * (NB * b + q);
                            if (g >= gf_lo && g < gf_hi) {
                                if (first) *reinterpret_cast<float4 *>(obase + 16ull * g) = v[q];
                                else asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};\n"
                                                  ::"l"(obase + 16ull * g), "f"(v[q].x), "f"(v[q].y), "f"(v[q].z), "f"(v[q].w) : "memory");
                            }
                        }
                    }
                    if (lane < 8) {   // lanes 0..3: the partial group below gf_lo; lanes 4..7: the one at gf_hi (the same group if gf_hi < gf_lo)
                        const int w = lane < 4 ? 4 * gf_lo - 4 + lane : 4 * gf_hi + lane - 4;
                        if (w >= w_lo && w < w_hi && (lane < 4 || gf_hi >= gf_lo)) {
                            if (first) *reinterpret_cast<float *>(obase + 4ull * w) = ep[w];
                            else asm volatile("red.global.add.f32 [%0], %1;\n" ::"l"(obase + 4ull * w), "f"(ep[w]) : "memory");
                        }
                    }
                }
            } else {
#pragma unroll 1
                for (int i = 0; i < TT / 32; ++i) put(i * 32 + lane);
            }
        }
    }
}

// u8 plans: the passes accumulate exact fp32 sums in place in the caller's int32 buffer (so that every
// pass can use the vector reduction); this turns the finished rows into int32, in place.
// VEC: rows start on 16-byte boundaries, a thread converts four consecutive samples with one 16-byte load and store.
template <bool VEC>
__global__ void __launch_bounds__(256) dedisp_f32_to_i32_inplace_kernel(int *__restrict__ out, long long out_stride, long long out_beam,
                                                                          long long nsamp_out, int d0) {
    const long long i = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * (VEC ? 4 : 1);
    if (i >= nsamp_out) return;
    int *pv = out + (size_t)blockIdx.z * out_beam + (size_t)(d0 + blockIdx.y) * out_stride + i;
    if (VEC && i + 3 < nsamp_out) {
        const float4 v = *reinterpret_cast<const float4 *>(pv);
        *reinterpret_cast<int4 *>(pv) = make_int4(__float2int_rn(v.x), __float2int_rn(v.y), __float2int_rn(v.z), __float2int_rn(v.w));
    } else {
        for (int q = 0; q < (VEC ? 4 : 1) && i + q < nsamp_out; ++q) pv[q] = __float2int_rn(__int_as_float(pv[q]));
    }
}

}  // namespace

// =====================================================================================
// host launch
// =====================================================================================
cudaError_t subband_upload(dedisp_plan *p) {
    SubbandGeom &sb = p->sb;
    if (!sb.ok) return cudaSuccess;
    std::vector<SbPassDev> tab(sb.passes.size());
    for (size_t g = 0; g < sb.passes.size(); ++g) {
        const SubbandPass &ps = sb.passes[g];
        bool last = true;                                 // no later pass covers this pass's DM blocks: the last sub-band of its range
        for (size_t h = g + 1; h < sb.passes.size(); ++h) last = last && sb.passes[h].blk_begin != ps.blk_begin;
        tab[g] = SbPassDev{ps.c_begin, ps.c_end, ps.blk_begin, ps.blk_end, ps.max_skew, ps.first ? 1 : 0, last ? 1 : 0, 0};
    }
    cudaError_t e = cudaMalloc(&sb.d_records, sb.records.size() * sizeof(uint64_t));
    if (e == cudaSuccess) e = cudaMemcpy(sb.d_records, sb.records.data(), sb.records.size() * sizeof(uint64_t), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc(&sb.d_meta, sb.meta.size() * sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMemcpy(sb.d_meta, sb.meta.data(), sb.meta.size() * sizeof(int32_t), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc(&sb.d_passes, tab.size() * sizeof(SbPassDev));
    if (e == cudaSuccess) e = cudaMemcpy(sb.d_passes, tab.data(), tab.size() * sizeof(SbPassDev), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc(&sb.d_skew, sb.skew.size() * sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMemcpy(sb.d_skew, sb.skew.data(), sb.skew.size() * sizeof(int32_t), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return e;
    switch (p->dtype) {
        case DEDISP_U8:
            e = sb.i16 ? cudaFuncSetAttribute(dedisp_subband_kernel<uint8_t, 6>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sb.smem_raw)
                       : cudaFuncSetAttribute(dedisp_subband_kernel<uint8_t, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sb.smem_raw);
            if (e == cudaSuccess && p->time_major && sb.i16) {
                e = cudaFuncSetAttribute(dedisp_subband_kernel<uint8_t, 7>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sb.smem);
                if (e == cudaSuccess) e = cudaFuncSetAttribute(dedisp_subband_kernel<uint8_t, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sb.smem);
                if (e == cudaSuccess) e = cudaFuncSetAttribute(dedisp_subband_kernel<uint8_t, 9>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sb.smem);
                if (e == cudaSuccess) e = cudaFuncSetAttribute(dedisp_subband_kernel<uint8_t, 10>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sb.smem);
            } else if (e == cudaSuccess && p->time_major) {   // time-major launches use the direct path's layout (no raw buffer)
                e = cudaFuncSetAttribute(dedisp_subband_kernel<uint8_t, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sb.smem);
                if (e == cudaSuccess) e = cudaFuncSetAttribute(dedisp_subband_kernel<uint8_t, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sb.smem);
                if (e == cudaSuccess) e = cudaFuncSetAttribute(dedisp_subband_kernel<uint8_t, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sb.smem);
                if (e == cudaSuccess) e = cudaFuncSetAttribute(dedisp_subband_kernel<uint8_t, 5>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sb.smem);
            }
            return e;
        case DEDISP_F16: return cudaFuncSetAttribute(dedisp_subband_kernel<__half, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sb.smem_raw);
        default: break;
    }
    e = cudaFuncSetAttribute(dedisp_subband_kernel<float, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sb.smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(dedisp_subband_kernel<float, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sb.smem_raw);
    return e;
}

void subband_free(dedisp_plan *p) {
    if (p->sb.d_records) cudaFree(p->sb.d_records);
    if (p->sb.d_meta) cudaFree(p->sb.d_meta);
    if (p->sb.d_skew) cudaFree(p->sb.d_skew);
    if (p->sb.d_passes) cudaFree(p->sb.d_passes);
    p->sb.d_records = nullptr;
    p->sb.d_meta = nullptr;
    p->sb.d_skew = nullptr;
    p->sb.d_passes = nullptr;
}

bool subband_smem_fits(const dedisp_plan *p) { return sb_smem_bytes(SB_CB, p->sb.max_nch + 1, dtype_esize(p->dtype), p->sb.i16) <= 227u * 1024u; }

// fp32 rows whose base and pitches are 16-byte aligned go straight into the ring; everything else takes the
// raw path (TMA of the raw bytes + conversion / realignment by the producer warps)
static bool sb_raw_path(const dedisp_plan *p, const void *d_in, long long in_stride, Batch b) {
    return p->dtype != DEDISP_F32 || ((uintptr_t)d_in & 15) != 0 || (in_stride & 3) != 0 || (b.n > 1 && (b.in_stride & 3) != 0);
}

// All passes in one launch? Ordered launches keep fp32 sums bit-reproducible (one add per address and
// pass, in pass order) and cost a launch gap plus a drained machine per pass; that only matters for plans
// cut into many short passes. u8 plans (exact, order-independent sums) merge below 48 channels per pass
// on average; fp plans only when the caller asked for it (dedisp_plan_set_pass_merge).
static bool sb_merge_passes(const dedisp_plan *p) {
    const size_t np = p->sb.passes.size();
    if (np < 2 || p->sb.nranges != 1) return false;
    if (p->dtype == DEDISP_U8) return (size_t)p->nchans <= 48 * np;
    return p->merge_fp_passes;
}

bool subband_merges(const dedisp_plan *p) { return sb_merge_passes(p); }

int subband_launches(const dedisp_plan *p, int resolved_kernel) {
    if (resolved_kernel != DEDISP_KERNEL_SUBBAND) return 1;
    const bool merged = sb_merge_passes(p);   // + a memset, which is not a kernel
    return (merged ? 1 : (int)p->sb.launch_begin.size() - 1) + (p->dtype == DEDISP_U8 ? 1 : 0);
}

cudaError_t launch_subband(dedisp_plan *p, const void *d_in, long long in_stride, long long nsamp_out, void *d_out,
                           long long out_stride, Batch b, cudaStream_t st, const SbRun &run) {
    const SubbandGeom &sb = p->sb;
    const long long nsamp_in = nsamp_out + p->maxshift;
    const int npass = (int)sb.passes.size();
    const int nlaunch = (int)sb.launch_begin.size() - 1;     // == npass for plans with one DM range
    const int pass_hi = run.pass_hi < 0 ? nlaunch : run.pass_hi;
    const int blk_lo = run.blk_lo, blk_hi = run.blk_hi < 0 ? sb.nblk : run.blk_hi;
    const bool whole = run.pass_lo == 0 && pass_hi == nlaunch && blk_lo == 0 && blk_hi == sb.nblk;
    SbArgs A;
    A.in_stride = in_stride;
    A.in_total = run.tm_bits ? nsamp_in : (long long)(p->nchans - 1) * in_stride + nsamp_in;   // time-major: rows (time samples) of in_stride bytes
    A.in_beam = b.in_stride;
    cudaError_t e;
    const bool raw = run.tm_bits == 0 && sb_raw_path(p, d_in, in_stride, b);
    A.in = d_in;
    A.out = d_out;
    A.out_stride = out_stride;
    A.out_beam = b.out_stride;
    A.nsamp_out = nsamp_out;
    A.out_vec4 = ((uintptr_t)d_out & 15) == 0 && (out_stride & 3) == 0 && (b.n == 1 || (b.out_stride & 3) == 0);
    A.records = sb.d_records;
    A.meta = reinterpret_cast<const int2 *>(sb.d_meta);
    A.skew = sb.d_skew;
    A.passes = sb.d_passes;
    A.ndm = p->ndm;
    A.nchans = p->nchans;
    A.nbeams = b.n;
    A.blk_lo = blk_lo;
    A.blk_hi = blk_hi;
    A.slot_chunks = sb.slot_chunks;
    A.raw_slot_bytes = sb.raw_slot_bytes;
    A.cb = raw ? sb.cb_raw : sb.cb;
    if (run.tm_bits && (A.cb != 16 || !p->time_major)) return cudaErrorInvalidValue;
    auto tiles_of = [&](const SubbandPass &ps) -> long long {
        const long long nb = std::min(blk_hi, ps.blk_end) - std::max(blk_lo, ps.blk_begin);
        return nb <= 0 ? 0 : nb * ((nsamp_out + ps.max_skew + sb.tile_t - 1) / sb.tile_t) * b.n;
    };
    auto launch = [&](long long tiles) -> cudaError_t {
        if (tiles <= 0) return cudaSuccess;
        if (tiles >= (1ll << 31)) return cudaErrorInvalidValue;
        const unsigned grid = (unsigned)std::min<long long>(tiles, std::max(1, p->sm_count));
        // u8 plans too accumulate fp32 sums (exact, checked at plan build) in place; converted after the last pass
        if (run.tm_bits && sb.i16) {
            if (run.tm_bits == 8) dedisp_subband_kernel<uint8_t, 7><<<grid, SB_THREADS, sb.smem, st>>>(A);
            else if (run.tm_bits == 4) dedisp_subband_kernel<uint8_t, 8><<<grid, SB_THREADS, sb.smem, st>>>(A);
            else if (run.tm_bits == 2) dedisp_subband_kernel<uint8_t, 9><<<grid, SB_THREADS, sb.smem, st>>>(A);
            else dedisp_subband_kernel<uint8_t, 10><<<grid, SB_THREADS, sb.smem, st>>>(A);
        }
        else if (run.tm_bits == 8) dedisp_subband_kernel<uint8_t, 2><<<grid, SB_THREADS, sb.smem, st>>>(A);
        else if (run.tm_bits == 4) dedisp_subband_kernel<uint8_t, 3><<<grid, SB_THREADS, sb.smem, st>>>(A);
        else if (run.tm_bits == 2) dedisp_subband_kernel<uint8_t, 4><<<grid, SB_THREADS, sb.smem, st>>>(A);
        else if (run.tm_bits == 1) dedisp_subband_kernel<uint8_t, 5><<<grid, SB_THREADS, sb.smem, st>>>(A);
        else if (!raw) dedisp_subband_kernel<float, 0><<<grid, SB_THREADS, sb.smem, st>>>(A);
        else if (sb.i16) dedisp_subband_kernel<uint8_t, 6><<<grid, SB_THREADS, sb.smem_raw, st>>>(A);
        else if (p->dtype == DEDISP_U8) dedisp_subband_kernel<uint8_t, 1><<<grid, SB_THREADS, sb.smem_raw, st>>>(A);
        else if (p->dtype == DEDISP_F16) dedisp_subband_kernel<__half, 1><<<grid, SB_THREADS, sb.smem_raw, st>>>(A);
        else dedisp_subband_kernel<float, 1><<<grid, SB_THREADS, sb.smem_raw, st>>>(A);
        return cudaGetLastError();
    };
    if (whole && sb_merge_passes(p)) {
        // all passes in ONE launch: out is zeroed, every pass adds with L2 reductions. Exact integers in
        // fp32 are order-independent, so u8 plans stay bit-reproducible; fp plans only take this path when
        // asked to (dedisp_plan_set_pass_merge), their sums then vary in the last bits.
        for (int bm = 0; bm < b.n; ++bm) {
            e = cudaMemset2DAsync((char *)d_out + (size_t)bm * b.out_stride * 4, (size_t)out_stride * 4, 0, (size_t)nsamp_out * 4, (size_t)p->ndm, st);
            if (e != cudaSuccess) return e;
        }
        long long tiles = 0;
        for (const SubbandPass &ps : sb.passes) tiles += tiles_of(ps);
        A.pass_lo = 0; A.pass_hi = npass; A.first = 0;
        e = launch(tiles);
        if (e != cudaSuccess) return e;
    } else {
        for (int i = run.pass_lo; i < pass_hi; ++i) {
            const int g = run.reverse ? nlaunch - 1 - i : i;          // launch g = passes [launch_begin[g], launch_begin[g + 1])
            A.pass_lo = sb.launch_begin[g]; A.pass_hi = sb.launch_begin[g + 1];
            A.first = sb.nranges == 1 ? i == 0 : run.reverse ? 3 : 2;   // one range: any order, the first launched pass stores; else per pass
            if (run.pass_ready) {   // dedisp_execute_host (one DM range): this pass's channel rows arrive on the copy stream
                e = cudaStreamWaitEvent(st, run.pass_ready[g], 0);
                if (e != cudaSuccess) return e;
            }
            long long tiles = 0;
            for (int q = A.pass_lo; q < A.pass_hi; ++q) tiles += tiles_of(sb.passes[q]);
            e = launch(tiles);
            if (e != cudaSuccess) return e;
        }
    }
    if (p->dtype == DEDISP_U8 && pass_hi == nlaunch) {   // last pass done for these rows
        const int d0 = std::min(p->ndm, blk_lo * SB_ROWS), d1 = std::min(p->ndm, blk_hi * SB_ROWS);
        for (int r0 = d0; r0 < d1; r0 += 32768) {   // grid.y <= 65535
            const int per = A.out_vec4 ? 1024 : 256;   // samples per CTA
            dim3 grid((unsigned)((nsamp_out + per - 1) / per), (unsigned)std::min(32768, d1 - r0), (unsigned)b.n);
            if (A.out_vec4) dedisp_f32_to_i32_inplace_kernel<true><<<grid, 256, 0, st>>>((int *)d_out, out_stride, b.out_stride, nsamp_out, r0);
            else dedisp_f32_to_i32_inplace_kernel<false><<<grid, 256, 0, st>>>((int *)d_out, out_stride, b.out_stride, nsamp_out, r0);
            e = cudaGetLastError();
            if (e != cudaSuccess) return e;
        }
    }
    return cudaSuccess;
}
