// fn_beam.cuh -- range sensing: exact first-hit distance of each beam on the bit-packed map.
//
// Operation: r = rho * inf{t : cell(o + t d) occupied}, capped at
// r_max, no hit => r_max; everything outside the map is occupied.
//
// The traversal is an exact grid walk organised by LINES instead of cells:
//   * the beam's dominant axis is "u", the other "w"; the packing whose bits run along u is used
//     (row-packed for |dx| >= |dy|, column-packed otherwise), so the beam stays in one line for
//     M = |du/dw| >= 1 cells before it crosses into the next line;
//   * line k is left at U_{k+1} = U_1 + k (+-M).  The crossing coordinate is carried as a double
//     D = 2^20 + 64 + U (+1 for beams running towards higher u): in [2^20, 2^21) a double is a 20.32
//     fixed-point number (ulp 2^-32 cell, far below the 1e-5 cell near-tie margin), its high word holds
//     floor(U) in the low bits, and "U += M" is ONE DADD on the otherwise idle fp64 pipe;
//   * per line ONE 64-bit window (two aligned 32-bit loads) is funnel-shifted by the low 5 bits of that
//     high word so that it ends (forward beams) or starts (backward beams) at the line's exit cell, and
//     ANDed with a per-beam constant mask of floor(M) + 2 bits that covers the cells the beam can have
//     visited in the line: non-zero = candidate hit.  Forward and backward beams run the SAME
//     instructions (the differences are per-lane constants), so a warp never serialises on direction;
//   * on a candidate the exact span [entry cell, exit cell] is rebuilt, the first occupied cell in
//     travel order is found with one clz/ctz, and the entry distance follows from the crossing
//     coordinates; a candidate outside the exact span (one extra cell behind the entry) resumes the walk;
//   * the map border is stored as occupied cells (fn_common.cuh), so leaving the map is an ordinary hit
//     (index -2) and the hot loop has no clipping at all.
// Beams within 1.9 deg of an axis (M >= 30.5, spans longer than one window) take a plain side path.
#pragma once
#include "fn_common.cuh"
#include <type_traits>

namespace fn {

// Address spaces for the packed map: staged in shared memory, or read through L1/L2.  The window
// address of a line is (line base) + 4 * (high word of D >> 5); the constant that D's exponent bits
// add to that offset (kExpOff) is subtracted from the line base once per beam, so no loop masks them off.
struct SmemSpace {
    using addr_t = uint32_t;                                     // shared-window byte address
    static __device__ __forceinline__ uint32_t ld(addr_t a) {
        uint32_t v;
        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a));
        return v;
    }
    static __device__ __forceinline__ uint32_t ld4(addr_t a) {
        uint32_t v;
        asm volatile("ld.shared.u32 %0, [%1+4];" : "=r"(v) : "r"(a));
        return v;
    }
    static __device__ __forceinline__ addr_t addb(addr_t a, int bytes) { return a + (uint32_t)bytes; }
    static __device__ __forceinline__ long long diffb(addr_t a, addr_t b) { return (long long)(int)(a - b); }
};
struct GlobalSpace {
    using addr_t = unsigned long long;                           // global byte address
    static __device__ __forceinline__ uint32_t ld(addr_t a) {
        uint32_t v;
        asm volatile("ld.global.nc.u32 %0, [%1];" : "=r"(v) : "l"(a));
        return v;
    }
    static __device__ __forceinline__ uint32_t ld4(addr_t a) {
        uint32_t v;
        asm volatile("ld.global.nc.u32 %0, [%1+4];" : "=r"(v) : "l"(a));
        return v;
    }
    static __device__ __forceinline__ addr_t addb(addr_t a, int bytes) { return a + (unsigned long long)(long long)bytes; }
    static __device__ __forceinline__ long long diffb(addr_t a, addr_t b) { return (long long)(a - b); }
};

template <class MS>
struct BeamMap {
    typename MS::addr_t base;        // start of the row copy (true address)
    int H, W, stride4R, stride4C;    // line strides in bytes
    unsigned rowBytes;               // size of the row copy = offset of the column copy
    unsigned mapBytes;               // both copies (instrumented kernels check every window against it)
    unsigned long long* oob;         // counter of windows outside [base, base + mapBytes) or NULL
};
// line index (row of the row copy / column of the column copy) of the origin's line
template <class MS>
__device__ __forceinline__ int origin_line(const BeamMap<MS>& bm, const BeamOrient& o, bool mx) {
    return mx ? (int)(o.line_off / (unsigned)bm.stride4R) - kLineGuard
              : (int)((o.line_off - bm.rowBytes) / (unsigned)bm.stride4C) - kLineGuard;
}

constexpr unsigned kExpOff = (kMagicHi >> 5) << 2;               // byte offset added by D's exponent bits
constexpr double kSlowSlope = 30.5;                              // spans of floor(M) + 2 <= 32 cells fit one window

__device__ __forceinline__ double rcp64h(double x) {             // MUFU.RCP64H: ~20-bit reciprocal
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    return r;
}
__device__ __forceinline__ unsigned hiw(double d) { return (unsigned)__double2hiint(d); }

struct BeamHit {
    float r;
    int hit;
};

// Entry distance of a hit along u -> range in metres: r = dU * (rho / |du|), the scale in fp32
// (ample: tolerance 1e-4 m on <= tens of metres).  Every path uses these two, so all agree bit for bit.
__device__ __forceinline__ float range_scale(double adu, float rho) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"((float)adu));
    return __fmul_rn(rho, r);
}
__device__ __forceinline__ float range_from_du(double dU, float scale) { return __fmul_rn((float)dU, scale); }

// ---- side path: beams nearly parallel to an axis (or exactly parallel: dw == 0).  Plain per-line walk
// over 32-bit words; at most T / 30 + 2 lines of up to T cells each.
template <class MS>
__device__ __noinline__ BeamHit cast_beam_slow(const BeamMap<MS> bm, const BeamOrient o, const bool mx,
                                               const double du, const double dw, const double M_in,
                                               const double T, const float rho, const float rmax) {
    // M_in = |du| / |dw| as the callers computed it (Newton-refined reciprocal, relative error ~2^-40: at most
    // ~1e-9 cell over a beam, far inside the 1e-5 cell near-tie margin); NaN or inf when dw == 0
    const double adu = fabs(du), adw = fabs(dw);
    const bool fu = du >= 0.0, fw = dw >= 0.0;
    const double ou = o.ouM - (kMagic + (double)kCellShift);
    const double f = fw ? 0.5 + o.h : 0.5 - o.h;
    const int Wu = mx ? bm.W : bm.H, Hw = mx ? bm.H : bm.W;
    const int stride4 = mx ? bm.stride4R : bm.stride4C;
    const double M = adw > 0.0 ? M_in : INFINITY;
    const double Tu = T * adu;                                    // travel along u at the range limit
    typename MS::addr_t line = MS::addb(bm.base, (int)o.line_off);
    int l = origin_line(bm, o, mx);
    double E = ou;                                                // entry coordinate of the current line
    for (int k = 0;; ++k) {
        double X = fu ? ou + (f + (double)k) * M : ou - (f + (double)k) * M;        // exit coordinate
        if (!(X > -1.0)) X = -0.5;                                // clamp into the frame cells (also NaN/inf)
        if (!(X < (double)Wu + 1.0)) X = (double)Wu + 0.5;
        const bool last = !(fabs(X - ou) < Tu);                   // the range limit lies in this line
        const int ce = __double2int_rd(E), cx = __double2int_rd(X);
        int c = ce, found = 0;
        if (fu) {
            while (c <= cx) {
                const int q = c + kCellShift;
                const uint32_t w = MS::ld(MS::addb(line, (q >> 5) << 2)) >> (q & 31);
                if (w) { c += __ffs(w) - 1; found = c <= cx; break; }
                c += 32 - (q & 31);
            }
        } else {
            while (c >= cx) {
                const int q = c + kCellShift;
                const uint32_t w = MS::ld(MS::addb(line, (q >> 5) << 2)) << (31 - (q & 31));
                if (w) { c -= __clz(w); found = c >= cx; break; }
                c -= (q & 31) + 1;
            }
        }
        if (found) {
            double dU;
            if (c == ce) dU = fabs(E - ou);                       // entered through the line boundary (or origin)
            else dU = fu ? (double)c - ou : ou - (double)(c + 1);
            if (!(dU < Tu)) break;
            BeamHit h;
            h.r = range_from_du(dU, range_scale(adu, rho));
            const bool outside = (unsigned)c >= (unsigned)Wu || (unsigned)l >= (unsigned)Hw;
            h.hit = outside ? -2 : (mx ? l * bm.W + c : c * bm.W + l);
            return h;
        }
        if (last) break;
        E = X;
        l += fw ? 1 : -1;
        line = MS::addb(line, fw ? stride4 : -stride4);
    }
    BeamHit h;
    h.r = rmax; h.hit = -1;
    return h;
}

// ---- one beam.  pose = the env's BeamPose (global memory), cs = (cos, sin) of the beam's body-frame angle.
// kAux additionally names the hit cell (linear index, -1 no hit, -2 outside the map) and counts 32-bit
// map words loaded.
template <class MS, bool kAux>
__device__ __forceinline__ float cast_beam(const BeamMap<MS>& bm, const BeamPose* __restrict__ pose,
                                           const double2 cs, const double T, const float rho, const float rmax,
                                           int* hit, uint32_t& words, const bool pair_lines = false) {
    const double2 pcs = *reinterpret_cast<const double2*>(&pose->c);
    const double dx = pcs.x * cs.x - pcs.y * cs.y, dy = pcs.y * cs.x + pcs.x * cs.y;
    const bool mx = fabs(dx) >= fabs(dy);                         // dominant axis is x
    const BeamOrient o = pose->o[mx ? 0 : 1];
    const double du = mx ? dx : dy, dw = mx ? dy : dx;
    const double adu = fabs(du), adw = fabs(dw);
    // slope M = |du / dw| >= 1: one Newton step on the 20-bit reciprocal (relative error ~2^-40)
    const double r0 = rcp64h(adw);
    const double r1 = fma(fma(-adw, r0, 1.0), r0, r0);
    const double M = adu * r1;
    if (!(M < kSlowSlope)) {                                      // also dw == 0 (M = inf or NaN)
        const BeamHit h = cast_beam_slow<MS>(bm, o, mx, du, dw, M, T, rho, rmax);
        if (kAux) { *hit = h.hit; words += 8; }
        return h.r;
    }
    const unsigned su = hiw(du) & 0x80000000u, sw = hiw(dw) & 0x80000000u;   // sign bits: set = backward
    const unsigned fu1 = (su >> 31) ^ 1u;                         // 1 for beams towards higher u
    // signed slope, distance f to the first line boundary (f = 0.5 + h forward in w, 0.5 - h backward)
    // (quantised to the 2^-32 grid of D, so that every later D +- Md is exact and path-independent)
    const double Mm = M + kMagic, Mq = Mm - kMagic;
    const double Md = __hiloint2double((int)(hiw(Mq) ^ su), __double2loint(Mq));
    const double f = __hiloint2double((int)(hiw(o.h) ^ sw), __double2loint(o.h)) + 0.5;
    // D_0 = 2^20 + 64 + U_1 (+ 1 forward): the "+ 1" is one unit of the integer field of the high word
    const double D0 = fma(f, Md, o.ouM);
    double D = __hiloint2double((int)(hiw(D0) + fu1), __double2loint(D0));
    // candidate mask: floor(M) + 2 cells ending (forward) / starting (backward) at the exit cell
    const unsigned sh = 30u - hiw(Mm);                    // low 5 bits = 30 - floor(M)
    const uint32_t mask = su ? __funnelshift_r(0xffffffffu, 0u, sh) : __funnelshift_l(0u, 0xffffffffu, sh);
    // lines: at most floor(T |dw|) + 2 (the frame stops every beam that would leave the map earlier)
    const int nl = __double2loint(fma(T, adw, 2.0 + 4503599627370496.0));
    const int stride4 = mx ? bm.stride4R : bm.stride4C;
    const int lstep = sw ? -stride4 : stride4;
    // forward beams read the window that ENDS at the exit cell: words (t >> 5) - 1 and t >> 5
    const typename MS::addr_t wb0 =
        MS::addb(bm.base, (int)(o.line_off - kExpOff) - (int)(fu1 << 2));
    float r = rmax;
    int hcell = -1;
    // A candidate in the line with crossing coordinate Dl and window base wl: rebuild the exact span
    // [entry cell ce, exit cell cx] (the origin cell replaces the entry cell in the first line).
    // Returns true when the traversal is over (hit within range, or first hit beyond the range).
    auto candidate = [&](const double Dl, const typename MS::addr_t wl, const uint32_t x) -> bool {
        const bool first = wl == wb0;
        const int cx = (int)(hiw(Dl) - kMagicHi - fu1);           // floor(U_{k+1}) + 64
        const double Dp = Dl - Md;
        const int ce = first ? o.cu0 + kCellShift : (int)(hiw(Dp) - kMagicHi - fu1);
        const unsigned n = 31u - (unsigned)abs(cx - ce);
        const uint32_t xe = x & (su ? __funnelshift_r(0xffffffffu, 0u, n) : __funnelshift_l(0u, 0xffffffffu, n));
        if (xe == 0u) return false;                               // the extra cell behind the entry: resume
        // first occupied cell in travel order: lowest bit forward, highest bit backward
        const int c = su ? cx + (31 - __clz(xe)) : cx - 31 + (__ffs(xe) - 1);
        double dU;
        if (c == ce) dU = first ? 0.0 : fabs(Dp - (o.ouM + (double)fu1));              // through the line boundary
        else dU = fabs((double)(c + (int)(su >> 31)) - (o.ouM - kMagic));              // through the cell's u-face
        if (dU < T * adu) {
            r = range_from_du(dU, range_scale(adu, rho));
            if (kAux) {
                const int k = (int)(MS::diffb(wl, wb0) / lstep);                       // lines crossed so far
                const int l0 = origin_line(bm, o, mx), lw = sw ? l0 - k : l0 + k, cu = c - kCellShift;
                const int Wu = mx ? bm.W : bm.H, Hw = mx ? bm.H : bm.W;
                const bool outside = (unsigned)cu >= (unsigned)Wu || (unsigned)lw >= (unsigned)Hw;
                hcell = outside ? -2 : (mx ? lw * bm.W + cu : cu * bm.W + lw);
            }
        }
        return true;                                              // later lines are farther away
    };
    if (std::is_same<MS, GlobalSpace>::value && !kAux && pair_lines) {
        // map read through L1/L2, long beams: two lines per trip, so that the (long-latency) loads of both overlap;
        // an odd line count is rounded up (one line beyond the range: its hits are rejected above)
        const typename MS::addr_t wend2 = MS::addb(wb0, (int)((unsigned)(nl - 1) | 1u) * lstep);
        typename MS::addr_t wb = MS::addb(wb0, lstep);            // the pair's second line
        const double Md2 = Md + Md;
        D += Md;
        for (;;) {
            const double Da = D - Md;
            const typename MS::addr_t wa = MS::addb(wb, -lstep);
            const uint32_t tha = hiw(Da), thb = hiw(D);
            const typename MS::addr_t aa = MS::addb(wa, (int)((tha >> 5) << 2)), ab = MS::addb(wb, (int)((thb >> 5) << 2));
            const uint32_t la = MS::ld(aa), ha = MS::ld4(aa), lb = MS::ld(ab), hb = MS::ld4(ab);
            const uint32_t xa = __funnelshift_r(la, ha, tha) & mask, xb = __funnelshift_r(lb, hb, thb) & mask;
            if (xa != 0u && candidate(Da, wa, xa)) break;
            if (xb != 0u && candidate(D, wb, xb)) break;
            if (wb == wend2) break;
            D += Md2;
            wb = MS::addb(wb, lstep + lstep);
        }
    } else {
        const typename MS::addr_t wend = MS::addb(wb0, (nl - 1) * lstep);
        typename MS::addr_t wb = wb0;
        for (;;) {
            uint32_t x;
            for (;;) {                                            // one window per line
                const uint32_t th = hiw(D);
                const typename MS::addr_t a = MS::addb(wb, (int)((th >> 5) << 2));
                if (kAux && bm.oob) {                            // self-check: the frame / pad / guard reasoning
                    const long long off = MS::diffb(a, bm.base);
                    if (off < 0 || off + 8 > (long long)bm.mapBytes) { atomicAdd(bm.oob, 1ull); x = 0u; break; }
                }
                x = __funnelshift_r(MS::ld(a), MS::ld4(a), th) & mask;
                if (kAux) words += 2;
                if (x != 0u || wb == wend) break;
                D += Md;
                wb = MS::addb(wb, lstep);
            }
            if (x == 0u || candidate(D, wb, x) || wb == wend) break;
            D += Md;
            wb = MS::addb(wb, lstep);
        }
    }
    if (kAux) *hit = hcell;
    return r;
}

// ---- one beam on the shared-memory map, production path.  Same arithmetic as cast_beam (all of it is
// exact fixed point, so both agree bit for bit), but the line is carried INSIDE D as well: the integer
// field of D (20 bits) holds the beam's BIT offset in its copy of the map, 8 * (byte offset of the line) + 64 + cell,
// and the per-line increment is +-M +- S (S = bits per line).  One DADD per line then advances the
// crossing coordinate and the line together, the window address is base + 4 * (high word >> 5), and the
// last line is recognised by the high word itself (line fields differ by >= S - 64 > 0): the hot loop
// needs no line pointer and no counter.  Two lines per trip (independent loads hide the shared-memory
// latency): 2 DADD, 2 x [SHF (word index), LEA (address), 2 LDS, SHF.W (window)], one LOP3 for
// ((xa | xb) & mask) != 0, one ISETP (last pair), BRA = 15 SASS instructions per two lines.
struct SmemGeo {
    uint32_t baseR, baseC;   // shared addresses of the row / column copy, - kExpOff
    float rho;
    int bitsR, bitsC;        // S: bits per line of the row / column copy
    float inv_bitsR, inv_bitsC;
};

__device__ __forceinline__ float cast_beam_smem(const BeamMap<SmemSpace>& bm, const SmemGeo& g,
                                                const BeamPose* __restrict__ pose, const double2 cs,
                                                const double T, const float rmax) {
    const double2 pcs = *reinterpret_cast<const double2*>(&pose->c);
    const double dx = pcs.x * cs.x - pcs.y * cs.y, dy = pcs.y * cs.x + pcs.x * cs.y;
    const bool mx = fabs(dx) >= fabs(dy);                         // dominant axis is x
    const BeamOrient o = pose->o[mx ? 0 : 1];
    const double du = mx ? dx : dy, dw = mx ? dy : dx;
    const double adu = fabs(du), adw = fabs(dw);
    const double r0 = rcp64h(adw);
    const double r1 = fma(fma(-adw, r0, 1.0), r0, r0);
    const double M = adu * r1;
    if (!(M < kSlowSlope)) return cast_beam_slow<SmemSpace>(bm, o, mx, du, dw, M, T, g.rho, rmax).r;
    const unsigned su = hiw(du) & 0x80000000u, sw = hiw(dw) & 0x80000000u;   // sign bits: set = backward
    const unsigned fu1 = (su >> 31) ^ 1u;
    const double Mm = M + kMagic, Mq = Mm - kMagic;
    const double Mu = __hiloint2double((int)(hiw(Mq) ^ su), __double2loint(Mq));      // +-M along u
    const double f = __hiloint2double((int)(hiw(o.h) ^ sw), __double2loint(o.h)) + 0.5;
    const int S = mx ? g.bitsR : g.bitsC;
    const double Sd = (double)S;                                  // (uniform: converted once per warp task)
    const double Md = Mu + __hiloint2double((int)(hiw(Sd) ^ sw), __double2loint(Sd)); // +-M +- S per line
    const double Md2 = Md + Md;
    // D of line 0 = 2^20 + bit offset of the origin's line + 64 + U_1 (+ 1 forward)
    const double D0f = fma(f, Mu, o.ouMS);
    const double D0 = __hiloint2double((int)(hiw(D0f) + fu1), __double2loint(D0f));
    const unsigned sh = 30u - hiw(Mm);
    const uint32_t mask = su ? __funnelshift_r(0xffffffffu, 0u, sh) : __funnelshift_l(0u, 0xffffffffu, sh);
    // P pairs of lines cover floor(T |dw|) + 2 lines; the frame stops beams that leave the map earlier
    const double Pd = fma(0.5 * T, adw, 1.5 + 4503599627370496.0) - 4503599627370496.0;
    double D = D0 - Md;                                           // rotated loop: the increments lead
    const uint32_t hend = hiw(fma(Pd, Md2, D));                   // high word of the last pair's second line
    const uint32_t base = (mx ? g.baseR : g.baseC) - (fu1 << 2);  // forward: the window ENDS at the exit cell
    const float scale = range_scale(adu, g.rho);
    const double Tu = T * adu;
    float r = rmax;
    for (;;) {
        uint32_t xa, xb;
        asm volatile(
            "{\n\t"
            ".reg .pred ph, pc;\n\t"
            ".reg .b32 j, a, L, H, lo, hia, hib, xo;\n\t"
            ".reg .f64 DA;\n\t"
            "FN_LOOP:\n\t"
            "add.f64 DA, %0, %3;\n\t"
            "add.f64 %0, %0, %4;\n\t"
            "mov.b64 {lo, hia}, DA;\n\t"
            "shr.u32 j, hia, 5;\n\t"
            "mad.lo.u32 a, j, 4, %5;\n\t"
            "ld.shared.u32 L, [a];\n\t"
            "ld.shared.u32 H, [a+4];\n\t"
            "shf.r.wrap.b32 %1, L, H, hia;\n\t"
            "mov.b64 {lo, hib}, %0;\n\t"
            "shr.u32 j, hib, 5;\n\t"
            "mad.lo.u32 a, j, 4, %5;\n\t"
            "ld.shared.u32 L, [a];\n\t"
            "ld.shared.u32 H, [a+4];\n\t"
            "shf.r.wrap.b32 %2, L, H, hib;\n\t"
            "or.b32 xo, %1, %2;\n\t"
            "and.b32 xo, xo, %7;\n\t"
            "setp.eq.u32 ph, xo, 0;\n\t"
            "setp.ne.and.u32 pc, hib, %6, ph;\n\t"
            "@pc bra FN_LOOP;\n\t"
            "}"
            : "+d"(D), "=r"(xa), "=r"(xb)
            : "d"(Md), "d"(Md2), "r"(base), "r"(hend), "r"(mask));
        xa &= mask;
        xb &= mask;
        // up to two candidate lines, in travel order: the pair's first line (D - Md), then its second (D)
        uint32_t x = xa;
        double Dl = D - Md;
        if (x == 0u) { x = xb; xb = 0u; Dl = D; }
        bool fin = false;
#pragma unroll 1
        while (x != 0u) {
            // exact span [entry cell ce, exit cell cx] of this line (origin cell in the first line)
            const uint32_t hl = hiw(Dl);
            const bool first = hl == hiw(D0);
            const int cx = (int)(hl - fu1);
            const double Dp = Dl - Mu;                            // entry crossing, same line field
            const int ce = first ? (int)hiw(o.ouMS) : (int)(hiw(Dp) - fu1);   // hiw(ouMS) = field of the origin cell
            const unsigned n = 31u - (unsigned)abs(cx - ce);
            const uint32_t xe = x & (su ? __funnelshift_r(0xffffffffu, 0u, n) : __funnelshift_l(0u, 0xffffffffu, n));
            if (xe != 0u) {
                // first occupied cell in travel order: highest bit backward, lowest bit forward
                const int c = cx - (int)(fu1 * 31u) + (31 - __clz(su ? xe : xe & (0u - xe)));
                // lines crossed: the integer fields of line k and line 0 differ by +-k S +- (cells along u)
                const int dq = sw ? (int)(hiw(D0) - hl) : (int)(hl - hiw(D0));
                const int k = __float2int_rd(fmaf((float)dq, mx ? g.inv_bitsR : g.inv_bitsC, 0.5f));
                const int lf = sw ? -k * S : k * S;                // line field of line k relative to line 0
                double dU;
                if (c == ce) dU = first ? 0.0 : fabs((Dp - (double)lf) - (o.ouMS + (double)fu1));
                else dU = fabs((double)(c + (int)(su >> 31) - lf - (int)kMagicHi) - (o.ouMS - kMagic));
                if (dU < Tu) r = range_from_du(dU, scale);
                fin = true;                                       // later lines are farther away
                break;
            }
            x = xb; xb = 0u; Dl = D;                              // the extra cell behind the entry: resume
        }
        if (fin || hiw(D) == hend) break;
    }
    return r;
}

struct BeamArgs {
    MapDev map;
    RobotDev robot;
    const BeamPose* poses;       // [N]
    const int* list;             // compacted env indices or NULL (= all envs)
    const int* count_dev;        // number of listed envs (device) or NULL
    int n_all;                   // number of envs when list == NULL
    float* out_ranges;           // [N][B]
    int* out_hit;                // [N][B] or NULL            (kAux only)
    float* ring_obs;             // ring base or NULL: also write ranges into the env's pending ring row
    unsigned long long ring_cap;
    const unsigned long long* ring_head;      // device: pending row of env e = (*ring_head + e) % ring_cap
    int ring_row;                // floats per ring row
    int count_words;             // (kAux only)
    int pair_lines;              // L1/L2 path: two lines per trip (pays off for long ranges)
    unsigned exp_off;            // = kExpOff, passed at run time: as a compile-time constant ptxas splits it over the
                                 // hot loop's address arithmetic (4 extra instructions per two lines) instead of
                                 // keeping base - kExpOff in one register
    unsigned* task_counter;      // next warp task; zeroed by the kernel that precedes the beam kernel
    float inv_bitsR, inv_bitsC;  // 1 / (bits per line) of the row / column copy (host-computed)
    int* flip_par_dev;           // fn_step's launch: clears done_count[*par ^ 1] and flips *par (see EnvArgs)
    int* done_count;
    const int* list_par_dev;     // or NULL; else list += (*list_par_dev ^ 1) * n_all, count_dev += (*list_par_dev ^ 1)
    unsigned long long* counters;
};

// One (env, beam) element: cast, store the range (and, instrumented, the hit cell; with a ring, the obs part
// of the env's pending ring row).  ring_head = slot of env 0's pending row.
template <class MS, bool kFast, bool kAux>
__device__ __forceinline__ void beam_element(const BeamArgs& a, const BeamMap<MS>& bm, const SmemGeo& geo,
                                             const double2* s_tab, const BeamPose* pose, const unsigned e, const unsigned j,
                                             const unsigned long long ring_head, uint32_t& words) {
    const int state = pose->state;
    float r = 0.0f;
    int hit = -2;
    if (state == 0) {
        if constexpr (kFast) r = cast_beam_smem(bm, geo, pose, s_tab[j], a.robot.T, a.robot.rmax);
        else r = cast_beam<MS, kAux>(bm, pose, s_tab[j], a.robot.T, a.map.rho, a.robot.rmax, &hit, words, a.pair_lines != 0);
    } else if (kAux) {
        if (state == 1) hit = origin_line(bm, pose->o[0], true) * a.map.W + pose->o[0].cu0;
        ++words;
    }
    const unsigned o = e * (unsigned)a.robot.B + j;                // n_envs * B < 2^31 (fn_sim_create)
    a.out_ranges[o] = r;
    if (kAux && a.out_hit) a.out_hit[o] = hit;
    if (a.ring_obs) {
        unsigned long long slot = ring_head + (unsigned long long)e;   // both < ring_cap
        if (slot >= a.ring_cap) slot -= a.ring_cap;
        a.ring_obs[slot * a.ring_row + j] = r;
    }
}

// Stages the beam table and (when `stage`) both packed copies of the map in shared memory: constants, so
// the kernels do this BEFORE their dependency wait, under the kernel that precedes them in the stream.
// The copy is done by the TMA engine: one thread arms an mbarrier with the byte count and issues 1-D bulk
// copies (cp.async.bulk, global -> shared), every thread then waits on the barrier's phase -- no registers,
// no LDG/STS instructions, and the SM's other CTA keeps its issue slots.  All threads of the CTA call; mbar =
// an 8-byte shared word of the caller, used once per launch.
__device__ __forceinline__ void stage_beam_constants(const BeamArgs& a, double2* s_tab, uint32_t* s_map,
                                                     const int mapWords, const bool stage, unsigned long long* mbar) {
    const uint32_t mb = (uint32_t)__cvta_generic_to_shared(mbar);
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mb));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const uint32_t tab_bytes = (uint32_t)a.robot.B * (uint32_t)sizeof(double2);
        const uint32_t map_bytes = stage ? ((uint32_t)mapWords * 4u) & ~15u : 0u;     // bulk copies move 16-byte units
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mb), "r"(tab_bytes + map_bytes) : "memory");
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     ::"r"((uint32_t)__cvta_generic_to_shared(s_tab)), "l"(a.robot.beam_cs), "r"(tab_bytes), "r"(mb) : "memory");
        const uint32_t dst = (uint32_t)__cvta_generic_to_shared(s_map);
        const uint8_t* src = reinterpret_cast<const uint8_t*>(a.map.row);              // row and col copies are contiguous
        for (uint32_t off = 0; off < map_bytes; off += 32768u) {
            const uint32_t sz = min(32768u, map_bytes - off);
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                         ::"r"(dst + off), "l"(src + off), "r"(sz), "r"(mb) : "memory");
        }
        if (stage) for (int i = (int)(map_bytes >> 2); i < mapWords; ++i) s_map[i] = __ldg(a.map.row + i);   // < 16 bytes
    }
    // phase 0 completes when the armed byte count has arrived
    uint32_t done = 0;
    for (int it = 0; it < (1 << 24) && !done; ++it)
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(mb) : "memory");
    if (!done) __trap();                                           // (never: a lost copy must not hang the device)
}

// The warps of the (persistent) grid take 32 consecutive (env, beam) pairs at a time: adjacent lanes =
// adjacent beams of one env, so a warp's loads mostly hit the same or neighbouring words (broadcast)
// and its lanes run similar trip counts.  kFast = production shared-memory traversal (cast_beam_smem).
template <class MS, bool kFast, bool kAux>
__device__ __forceinline__ void run_beam_tasks(const BeamArgs& a, const BeamMap<MS>& bm, const SmemGeo& geo,
                                               const double2* s_tab, const int n_env, const unsigned total,
                                               const unsigned long long ring_head,     // slot of env 0's pending ring row
                                               const unsigned warp0, const unsigned nwarps,  // this warp's place among the
                                               const bool has_static = true) {         // warps that share the static part
    const int B = a.robot.B;
    const int lane = threadIdx.x & 31;
    const unsigned ntasks = (total + 31u) >> 5;
    uint32_t words = 0, rays = 0;
    // Beams differ in length by an order of magnitude, and a purely static split leaves ~15 % of the SM
    // time idle at the end of the launch.  So: the first 3/4 of each warp's share is static (round r ->
    // task warp0 + r * nwarps, no atomics), the rest is handed out dynamically, one atomic per warp
    // task, fetched one task ahead so that its latency is hidden.
    // (has_static = false: a warp that arrives late -- fn_step_split.cuh -- takes pool tasks only)
    const unsigned static_rounds = max(1u, ((ntasks / nwarps) * 3u) >> 2);
    const unsigned dyn_base = static_rounds * nwarps;
    const bool dynamic = dyn_base < ntasks;                        // (short launches are static only)
    const unsigned long long invB = ~0ull / (unsigned long long)B + 1ull;     // floor(2^64 / B) + 1
    unsigned round = 0;
    unsigned task = warp0;
    if (!has_static) {
        round = static_rounds;
        task = ntasks;
        if (dynamic && lane == 0) task = dyn_base + atomicAdd(a.task_counter, 1u);
        task = __shfl_sync(0xffffffffu, task, 0);
    }
    while (task < ntasks) {
        unsigned next = ntasks;
        ++round;
        if (round < static_rounds) next = warp0 + round * nwarps;
        else if (dynamic && lane == 0) next = dyn_base + atomicAdd(a.task_counter, 1u);
        // (listed env, beam) of this lane's element idx = 32 task + lane
        const unsigned idx = (task << 5) + lane;
        const unsigned le = (unsigned)__umul64hi((unsigned long long)idx, invB);     // idx / B, exact for idx < 2^32
        const unsigned j = idx - le * (unsigned)B;
        if (le < (unsigned)n_env) {
            const unsigned e = a.list ? (unsigned)a.list[le] : le;
            beam_element<MS, kFast, kAux>(a, bm, geo, s_tab, a.poses + e, e, j, ring_head, words);
            ++rays;
        }
        task = __shfl_sync(0xffffffffu, next, 0);
    }
    // counters: one atomic per warp
    for (int o = 16; o > 0; o >>= 1) {
        rays += __shfl_xor_sync(0xffffffffu, rays, o);
        if (kAux) words += __shfl_xor_sync(0xffffffffu, words, o);
    }
    if (lane == 0) {
        atomicAdd(&a.counters[kRays], (unsigned long long)rays);
        if (kAux && a.count_words) atomicAdd(&a.counters[kWords], (unsigned long long)words);
    }
}

// Persistent kernel (grid = SMs x resident CTAs).  kSmem: each CTA stages both packed copies of the map
// and the beam table in shared memory -- constants, so this happens BEFORE the dependency wait, under
// the env-step / reset kernel that precedes it in the stream.
// kAux = instrumented variant: hit-cell output, map-word counter.
template <bool kSmem, bool kAux>
__global__ void __launch_bounds__(512, 2) beam_kernel(BeamArgs a) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    const int B = a.robot.B;
    constexpr bool stage = kSmem;
    const int mapWords = (a.map.H + 2 * kLineGuard) * a.map.strideR + (a.map.W + 2 * kLineGuard) * a.map.strideC;
    double2* s_tab = reinterpret_cast<double2*>(smem_raw);
    uint32_t* s_map = reinterpret_cast<uint32_t*>(smem_raw + (size_t)B * sizeof(double2));
    __shared__ __align__(8) unsigned long long s_mbar;
    stage_beam_constants(a, s_tab, s_map, mapWords, stage, &s_mbar);
    __syncthreads();
    griddep_wait();                                                // poses / list / count come from the previous kernel
    griddep_launch_dependents();
    if (a.flip_par_dev && blockIdx.x == 0 && threadIdx.x == 0) {
        const int p = *a.flip_par_dev;
        a.done_count[p ^ 1] = 0;
        *a.flip_par_dev = p ^ 1;
    }
    if (a.list_par_dev) { const int q = *a.list_par_dev ^ 1; a.list += (size_t)q * a.n_all; a.count_dev += q; }
    const int n_env = a.count_dev ? *a.count_dev : a.n_all;
    const unsigned total = (unsigned)n_env * (unsigned)B;
    const unsigned long long ring_head = a.ring_obs ? *a.ring_head : 0ull;
    const unsigned warp0 = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const unsigned nwarps = gridDim.x * (blockDim.x >> 5);

    SmemGeo geo;
    geo.baseR = geo.baseC = 0; geo.rho = a.map.rho; geo.bitsR = a.map.strideR << 5; geo.bitsC = a.map.strideC << 5;
    geo.inv_bitsR = a.inv_bitsR; geo.inv_bitsC = a.inv_bitsC;
    const unsigned rowBytes = (unsigned)(a.map.H + 2 * kLineGuard) * (unsigned)(a.map.strideR << 2);
    if (stage) {
        BeamMap<SmemSpace> bm;
        bm.base = (uint32_t)__cvta_generic_to_shared(s_map);
        bm.H = a.map.H; bm.W = a.map.W; bm.stride4R = a.map.strideR << 2; bm.stride4C = a.map.strideC << 2;
        bm.rowBytes = rowBytes; bm.mapBytes = (unsigned)mapWords * 4u; bm.oob = a.counters + kOobLoads;
        geo.baseR = bm.base - a.exp_off; geo.baseC = geo.baseR + rowBytes;
        run_beam_tasks<SmemSpace, !kAux, kAux>(a, bm, geo, s_tab, n_env, total, ring_head, warp0, nwarps);
    } else {
        BeamMap<GlobalSpace> bm;
        bm.base = (unsigned long long)__cvta_generic_to_global(a.map.row);
        bm.H = a.map.H; bm.W = a.map.W; bm.stride4R = a.map.strideR << 2; bm.stride4C = a.map.strideC << 2;
        bm.rowBytes = rowBytes; bm.mapBytes = (unsigned)mapWords * 4u; bm.oob = a.counters + kOobLoads;
        run_beam_tasks<GlobalSpace, false, kAux>(a, bm, geo, s_tab, n_env, total, ring_head, warp0, nwarps);
    }
}

}  // namespace fn
