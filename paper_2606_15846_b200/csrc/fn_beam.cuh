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

// Direction of a beam = heading (pcs = cos, sin) rotated by the beam's body-frame angle (cs).  The rounding order
// is spelled out: left to the compiler, "a * b - c * d" contracts into an fma around either product, and two
// kernels that chose differently disagree in the last bit of a range now and then.  The case that did occur (one
// range in ~10^9, found by the 1000-step run): the slope M = |du| * r1 contracted with the "+ 2^20" that puts it on
// the grid of D in the instrumented kernel only -- one rounding instead of two, M differing by 2^-32 -- so M is
// rounded by explicit __dmul_rn / __dadd_rn in every kernel.
__device__ __forceinline__ double beam_dir_x(const double2 pcs, const double2 cs) { return fma(pcs.x, cs.x, -__dmul_rn(pcs.y, cs.y)); }
__device__ __forceinline__ double beam_dir_y(const double2 pcs, const double2 cs) { return fma(pcs.y, cs.x, __dmul_rn(pcs.x, cs.y)); }

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
    const int lstep = fw ? stride4 : -stride4;
    int l = origin_line(bm, o, mx);
    BeamHit h;
    h.r = rmax; h.hit = -1;
    // ONE flat loop whose trip is "one 32-bit word of the current line" (a walk nested as lines x words made
    // the lanes of a warp drift apart: every lane then ran its own inner loop alone)
    double E = ou, X;                                             // entry / exit coordinate of the current line
    int k = 0, ce, cx, c;
    bool last;
    auto enter_line = [&]() {
        X = fma(fu ? f + (double)k : -(f + (double)k), M, ou);     // (one rounding, spelled out: see beam_dir_x)
        if (!(X > -1.0)) X = -0.5;                                // clamp into the frame cells (also NaN/inf)
        if (!(X < (double)Wu + 1.0)) X = (double)Wu + 0.5;
        last = !(fabs(X - ou) < Tu);                              // the range limit lies in this line
        ce = __double2int_rd(E); cx = __double2int_rd(X);
        c = ce;
    };
    enter_line();
    for (;;) {
        const int q = c + kCellShift;
        uint32_t w = MS::ld(MS::addb(line, (q >> 5) << 2));
        int cn;
        bool found;
        if (fu) { w >>= (q & 31); cn = w ? c + __ffs(w) - 1 : c + 32 - (q & 31); found = w != 0u && cn <= cx; }
        else { w <<= 31 - (q & 31); cn = w ? c - __clz(w) : c - (q & 31) - 1; found = w != 0u && cn >= cx; }
        if (found) {                                              // first occupied cell of the line's span
            c = cn;
            double dU;
            if (c == ce) dU = fabs(E - ou);                       // entered through the line boundary (or origin)
            else dU = fu ? (double)c - ou : ou - (double)(c + 1);
            if (dU < Tu) {
                h.r = range_from_du(dU, range_scale(adu, rho));
                const bool outside = (unsigned)c >= (unsigned)Wu || (unsigned)l >= (unsigned)Hw;
                h.hit = outside ? -2 : (mx ? l * bm.W + c : c * bm.W + l);
            }
            break;
        }
        if (w == 0u && (fu ? cn <= cx : cn >= cx)) { c = cn; continue; }   // next word of the same line
        if (last) break;                                          // the line's span is free
        E = X; ++k;
        l += fw ? 1 : -1;
        line = MS::addb(line, lstep);
        enter_line();
    }
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
    const double dx = beam_dir_x(pcs, cs), dy = beam_dir_y(pcs, cs);
    const bool mx = fabs(dx) >= fabs(dy);                         // dominant axis is x
    const BeamOrient o = pose->o[mx ? 0 : 1];
    const double du = mx ? dx : dy, dw = mx ? dy : dx;
    const double adu = fabs(du), adw = fabs(dw);
    // slope M = |du / dw| >= 1: one Newton step on the 20-bit reciprocal (relative error ~2^-40)
    const double r0 = rcp64h(adw);
    const double r1 = fma(fma(-adw, r0, 1.0), r0, r0);
    const double M = __dmul_rn(adu, r1);                         // (rounded here: see beam_dir_x)
    if (!(M < kSlowSlope)) {                                      // also dw == 0 (M = inf or NaN)
        const BeamHit h = cast_beam_slow<MS>(bm, o, mx, du, dw, M, T, rho, rmax);
        if (kAux) { *hit = h.hit; words += 8; }
        return h.r;
    }
    const unsigned su = hiw(du) & 0x80000000u, sw = hiw(dw) & 0x80000000u;   // sign bits: set = backward
    const unsigned fu1 = (su >> 31) ^ 1u;                         // 1 for beams towards higher u
    // signed slope, distance f to the first line boundary (f = 0.5 + h forward in w, 0.5 - h backward)
    // (quantised to the 2^-32 grid of D, so that every later D +- Md is exact and path-independent)
    const double Mm = __dadd_rn(M, kMagic), Mq = __dadd_rn(Mm, -kMagic);   // (never fma(adu, r1, kMagic): one rounding less)
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

// ---- production path on the shared-memory map (fn_beam_fast below).  Same arithmetic as cast_beam (all of
// it is exact fixed point, so both agree bit for bit), but the line is carried INSIDE D as well: the integer
// field of D (20 bits) holds the beam's BIT offset in its copy of the map, 8 * (byte offset of the line) + 64 + cell,
// and the per-line increment is +-M +- S (S = bits per line).  One DADD per line then advances the
// crossing coordinate and the line together, the window address is base + 4 * (high word >> 5), and the
// last line is recognised by the high word itself (line fields differ by >= S - 64 > 0): the hot loop
// needs no line pointer and no counter.  Two lines per trip (independent loads hide the shared-memory
// latency): 2 DADD, 2 x [SHF (word index), LEA (address), 2 LDS, SHF.W (window)], one LOP3 for
// ((xa | xb) & mask) != 0, one ISETP (last pair), BRA = 15 SASS instructions per two lines.
//
// Everything a beam needs besides its own direction sits in a 128-byte slot of shared memory owned by the
// warp (FastSlot): the heading and, per dominant axis, the origin (h, ouMS) and the constants of the copy.
// A beam selects its axis by ONE address and reads 16-byte records at fixed offsets from it -- no global
// pointers, no 64-bit address arithmetic and nothing to rematerialise in the per-beam code.
struct __align__(16) FastAxis {                                  // 48 bytes
    double h, ouMS;          // BeamOrient::h, ::ouMS of the env being cast (rewritten per task)
    double Sd;               // S: bits per line of the copy, as a double
    uint32_t base;           // shared address of the copy - kExpOff
    uint32_t half_S;         // S / 2
    uint32_t inv_magic;      // ceil(2^32 / S): lines crossed k = umulhi(field difference + S / 2, inv_magic), exact
    uint32_t S;
    uint32_t base_c;         // shared address of the coarse copy - kExpOff (kCoarse)
    uint32_t par;            // parity of the physical line of the origin (rewritten per task; kCoarse)
};
struct __align__(16) FastSlot {                                  // 128 bytes per warp
    double pc, ps;           // cos / sin of the heading (rewritten per task)
    FastAxis ax[2];          // [0] u = x (row copy), [1] u = y (column copy)
    uint32_t pad_[4];
};
constexpr int kNearQueue = 64;                                   // per warp: deferred near-axis beams

__device__ __forceinline__ double xor_hi(double v, unsigned m) { return __hiloint2double((int)(hiw(v) ^ m), __double2loint(v)); }
__device__ __forceinline__ double add_hi(double v, unsigned k) { return __hiloint2double((int)(hiw(v) + k), __double2loint(v)); }
// a value the compiler must keep in its register (it would otherwise rebuild shared addresses per use)
__device__ __forceinline__ uint32_t opaque(uint32_t v) { asm volatile("mov.b32 %0, %0;" : "+r"(v)); return v; }
__device__ __forceinline__ double2 lds_d2(uint32_t addr) {
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}

// The hot loop: two lines (kCoarse: two PAIRS of lines) per trip.  D = crossing coordinate of the line before
// the trip's first one; on exit D belongs to the trip's second line, xa / xb are the two (unmasked) windows.
__device__ __forceinline__ void fast_loop(double& D, uint32_t& xa, uint32_t& xb, const double Md, const double Md2,
                                          const uint32_t base, const uint32_t hend, const uint32_t mask) {
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
}
// the window of the line with crossing coordinate Dl (base = the copy's base, - 4 for forward beams)
__device__ __forceinline__ uint32_t fast_window(const uint32_t base, const double Dl) {
    const uint32_t h = hiw(Dl), a = base + ((h >> 5) << 2);
    return __funnelshift_r(SmemSpace::ld(a), SmemSpace::ld4(a), h);
}

// One beam per lane.  slot = shared address of the warp's FastSlot; tab = shared address of the beam's
// (cos, sin) entry.  near = the beam is too close to an axis for a 32-bit window (M >= 30.5; with the coarse
// level 2 M >= 30.5): not cast here, the caller defers it (fast_chunk / fast_drain).
// kCoarse: the hot loop walks the coarse copy, one window per PAIR of lines (the pairs are aligned in the map, so
// a beam's first pair may hold one of its lines only); a non-empty window sends the pair's two fine lines through
// the same tests as without the coarse level, in travel order, so that both variants resolve the same line with
// the same crossing coordinates (every coordinate is D0 plus exact multiples of M and S): identical results.
template <bool kCoarse>
__device__ __forceinline__ float cast_beam_fast(const uint32_t slot, const uint32_t tab, const double T,
                                                const double half_T, const float rho, const float rmax, bool& near) {
    const double2 cs = lds_d2(tab), pcs = lds_d2(slot);
    const double dx = beam_dir_x(pcs, cs), dy = beam_dir_y(pcs, cs);
    const bool mx = fabs(dx) >= fabs(dy);                         // dominant axis is x
    const double du = mx ? dx : dy, dw = mx ? dy : dx;
    const double adw = __hiloint2double((int)(hiw(dw) & 0x7fffffffu), __double2loint(dw));
    const double r0 = rcp64h(adw);
    const double r1 = fma(fma(-adw, r0, 1.0), r0, r0);
    const double M = __dmul_rn(fabs(du), r1);                     // (rounded here: see beam_dir_x)
    near = !(M < (kCoarse ? 0.5 * kSlowSlope : kSlowSlope));      // also dw == 0 (M = inf or NaN)
    float r = rmax;
    // (a near-axis lane stays with the warp: it walks one trip of a harmless beam of slope 1 and its result is
    // dropped, so that the whole warp reaches the resolution below converged)
    const double Mc = near ? 1.0 : M;
    const uint32_t ax = slot + (mx ? 16u : 64u);                  // the axis record
    const double2 hq = lds_d2(ax);                                // (h, ouMS)
    double Sd;
    uint32_t base;
    asm volatile("ld.shared.f64 %0, [%1+16];" : "=d"(Sd) : "r"(ax));
    asm volatile("ld.shared.u32 %0, [%1+24];" : "=r"(base) : "r"(ax));
    const unsigned su = hiw(du) & 0x80000000u, sw = hiw(dw) & 0x80000000u;   // sign bits: set = backward
    const unsigned fu1 = (su >> 31) ^ 1u;
    const double Mm = __dadd_rn(Mc, kMagic), Mq = __dadd_rn(Mm, -kMagic);   // M on the 2^-32 grid of D
    const double Mu = xor_hi(Mq, su);                             // +-M along u
    const double f = xor_hi(hq.x, sw) + 0.5;                      // distance to the first line boundary, in lines
    const double Md = Mu + xor_hi(Sd, sw);                        // +-M +- S per line
    // D of line 0 = 2^20 + bit offset of the origin's line + 64 + U_1 (+ 1 forward)
    const double D0 = add_hi(fma(f, Mu, hq.y), fu1);
    const unsigned sh = 30u - hiw(Mm);                            // candidate mask of a line: floor(M) + 2 cells
    const uint32_t mask = su ? __funnelshift_r(0xffffffffu, 0u, sh) : __funnelshift_l(0u, 0xffffffffu, sh);
    base -= fu1 << 2;                                             // forward: the window ENDS at the exit cell
    const uint32_t h0 = hiw(D0), hc0 = hiw(hq.y);                 // fields of line 0 and of the origin cell
    double Dh = 0.0;                                              // the hit line's D and exact window (xh != 0: hit)
    uint32_t xh = 0u;
    // exact span [entry cell ce, exit cell cx] of the line with crossing coordinate Dl (origin cell in line 0)
    auto exact = [&](const uint32_t x, const double Dl) -> uint32_t {
        const uint32_t hl = hiw(Dl);
        const int cx = (int)(hl - fu1);
        const int ce = hl == h0 ? (int)hc0 : (int)(hiw(Dl - Mu) - fu1);
        const unsigned n = 31u - (unsigned)abs(cx - ce);
        return x & (su ? __funnelshift_r(0xffffffffu, 0u, n) : __funnelshift_l(0u, 0xffffffffu, n));
    };
    if constexpr (!kCoarse) {
        const double Md2 = Md + Md;
        // P pairs of lines cover floor(T |dw|) + 2 lines; the frame stops beams that leave the map earlier
        const double Pd = near ? 1.0 : fma(half_T, adw, 1.5 + 4503599627370496.0) - 4503599627370496.0;
        double D = D0 - Md;                                       // rotated loop: the increments lead
        const uint32_t hend = hiw(fma(Pd, Md2, D));               // high word of the last pair's second line
        for (;;) {
            uint32_t xa, xb;
            fast_loop(D, xa, xb, Md, Md2, base, hend, mask);
            // up to two candidate lines, in travel order: the pair's first line (D - Md), then its second (D).
            // Only the exact-span test runs here (per loop exit); the hit itself is resolved once, below.
            uint32_t x = xa & mask, xn = xb & mask;
            double Dl = D - Md;
            if (x == 0u) { x = xn; xn = 0u; Dl = D; }
#pragma unroll 1
            while (x != 0u) {
                const uint32_t xe = exact(x, Dl);
                if (xe != 0u) { xh = xe; Dh = Dl; break; }
                x = xn; xn = 0u; Dl = D;                          // the extra cell behind the entry: next line / resume
            }
            if (xh != 0u || hiw(D) == hend) break;
        }
    } else {
        uint32_t base_c, par;                                     // coarse copy; parity of the origin's physical line
        asm volatile("ld.shared.v2.u32 {%0, %1}, [%2+40];" : "=r"(base_c), "=r"(par) : "r"(ax));
        const unsigned q = sw ? par : par ^ 1u;                   // 1: the first pair holds two lines of the beam
        const double Mdc = Md + Md, Mdc2 = Mdc + Mdc;             // per pair: +-2 M +- 2 S
        // D of pair 0 = exit crossing of its last line, with the bit offset of its even line
        const double D0c = (D0 + (q ? Mu : 0.0)) - (par ? Sd : 0.0);
        const unsigned shc = 30u - hiw(Mm + Mq);                  // candidate mask of a pair: floor(2 M) + 2 cells
        const uint32_t maskc = su ? __funnelshift_r(0xffffffffu, 0u, shc) : __funnelshift_l(0u, 0xffffffffu, shc);
        // P trips of two pairs cover floor(T |dw|) + 2 lines from any alignment
        const double Pd = near ? 1.0 : fma(0.5 * half_T, adw, 2.0 + 4503599627370496.0) - 4503599627370496.0;
        double D = D0c - Mdc;
        const uint32_t hend = hiw(fma(Pd, Mdc2, D));
        base_c -= fu1 << 2;
        const uint32_t h0c = hiw(D0c);
        const double SA = sw ? Sd : 0.0, SB = sw ? 0.0 : Sd;      // line field of the pair's first / second line in travel order
        for (;;) {
            uint32_t xa, xb;
            fast_loop(D, xa, xb, Mdc, Mdc2, base_c, hend, maskc);
            uint32_t x = xa & maskc, xn = xb & maskc;
            double Dg = D - Mdc;
            if (x == 0u) { x = xn; xn = 0u; Dg = D; }
#pragma unroll 1
            while (x != 0u) {                                     // a non-empty pair: its two fine lines
                const double DA = (Dg - Mu) + SA, DB = Dg + SB;
                uint32_t wA = fast_window(base, DA) & mask;
                const uint32_t wB = fast_window(base, DB) & mask;
                if (hiw(Dg) == h0c && q == 0u) wA = 0u;           // (the first pair's other line lies behind the origin)
                if (wA != 0u) { const uint32_t xe = exact(wA, DA); if (xe != 0u) { xh = xe; Dh = DA; } }
                if (xh == 0u && wB != 0u) { const uint32_t xe = exact(wB, DB); if (xe != 0u) { xh = xe; Dh = DB; } }
                if (xh != 0u) break;
                x = xn; xn = 0u; Dg = D;
            }
            if (xh != 0u || hiw(D) == hend) break;
        }
    }
    __syncwarp();                                                 // resolve all hits of the warp together
    if (xh != 0u) {                                               // later lines are farther away
        // Everything below is in the hit line's own bit-offset units (high words of D's).  The hit cell c is the
        // first occupied cell of the exact window in travel order (highest bit backward, lowest bit forward); the beam
        // enters it through the line boundary when c is the line's entry cell (the cell of the entry crossing
        // Dp = Dh - M: never so in line 0, whose entry cell is the free origin cell), else through the cell's u-face,
        // whose coordinate is c + 1 in D's convention for both directions (forward D's carry + 1).
        const uint32_t hl = hiw(Dh);
        const double Dp = Dh - Mu;                                // entry crossing, same line field
        const uint32_t c = hl - (fu1 << 5) + (uint32_t)(31 - __clz(su ? xh : xh & (0u - xh)));
        const bool ent = c == hiw(Dp) - fu1;
        // lines crossed: the integer fields of line k and line 0 differ by +-k S +- (cells along u)
        uint32_t half_S, inv_magic, S;
        asm volatile("ld.shared.u32 %0, [%1+28];" : "=r"(half_S) : "r"(ax));
        asm volatile("ld.shared.v2.u32 {%0, %1}, [%2+32];" : "=r"(inv_magic), "=r"(S) : "r"(ax));
        const int sgw = sw ? -1 : 1;
        const uint32_t k = __umulhi((hl - h0) * (uint32_t)sgw + half_S, inv_magic);
        const uint32_t lf = k * S * (uint32_t)sgw;                // line field of line k relative to line 0
        // entry distance along u = | hit coordinate - origin |, both with line 0's field
        const double a = __hiloint2double((int)((ent ? hiw(Dp) : c + 1u) - lf), ent ? __double2loint(Dp) : 0);
        const double dU = fabs(a - add_hi(hq.y, fu1));
        const double adu = fabs(du);
        if (dU < T * adu) r = range_from_du(dU, range_scale(adu, rho));
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
    float* out_ranges;           // [N][out_stride]: this launch writes columns out_off .. out_off + B - 1 of a row
    int* out_hit;                // the same layout, or NULL  (kAux only)
    unsigned out_stride, out_off;  // (a robot with several sensors: one launch per sensor, B = that sensor's beams)
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
    unsigned inv_magicR, inv_magicC;   // ceil(2^32 / bits per line) of the row / column copy (FastOrient::inv_magic)
    double half_T;               // 0.5 * robot.T
    int chunk_rounds, nchunk;    // production kernel: a warp task of the static part = chunk_rounds x 32 consecutive
                                 // beams of one env, nchunk such tasks per env (host: fast_chunking); the tasks of the
                                 // dynamic part are single rounds of 32 beams
    unsigned inv_nchunk, inv_rounds;   // fast_magic(nchunk), fast_magic(rounds per env): t / d = umulhi(t, magic), or 0
    int* flip_par_dev;           // fn_step's launch: clears done_count[*par ^ 1] and flips *par (see EnvArgs)
    int* done_count;
    const int* list_par_dev;     // or NULL; else list += (*list_par_dev ^ 1) * n_all, count_dev += (*list_par_dev ^ 1)
    unsigned long long* counters;
};

// One (env, beam) element of the instrumented / L2-path kernels: cast, store the range (and, instrumented, the
// hit cell; with a ring, the obs part of the env's pending ring row).  ring_head = slot of env 0's pending row.
template <class MS, bool kAux>
__device__ __forceinline__ void beam_element(const BeamArgs& a, const BeamMap<MS>& bm,
                                             const double2* s_tab, const BeamPose* pose, const unsigned e, const unsigned j,
                                             const unsigned long long ring_head, uint32_t& words) {
    const int state = pose->state;
    float r = 0.0f;
    int hit = -2;
    if (state == 0) {
        r = cast_beam<MS, kAux>(bm, pose, s_tab[j], a.robot.T, a.map.rho, a.robot.rmax, &hit, words, a.pair_lines != 0);
    } else if (kAux) {
        if (state == 1) hit = origin_line(bm, pose->o[0], true) * a.map.W + pose->o[0].cu0;
        ++words;
    }
    const unsigned o = e * a.out_stride + a.out_off + j;           // n_envs * row length < 2^31 (fn_sim_create)
    a.out_ranges[o] = r;
    if (kAux && a.out_hit) a.out_hit[o] = hit;
    if (a.ring_obs) {
        unsigned long long slot = ring_head + (unsigned long long)e;   // both < ring_cap
        if (slot >= a.ring_cap) slot -= a.ring_cap;
        a.ring_obs[slot * a.ring_row + a.out_off + j] = r;
    }
}

// ---- production kernel: warp tasks of chunk_rounds x 32 consecutive beams of ONE env.  What depends on the env
// only (list entry, pose, output rows) is done once per task; near-axis beams are not cast in place (a
// divergent walk over single words) but queued per warp and cast 32 at a time (fast_drain).
template <int kWarps>                                              // warps per CTA
struct FastShared {
    FastSlot slot[kWarps];
    uint32_t queue[kWarps][kNearQueue];                            // deferred beams: output offsets e * B + j
};
// launch shape of the production kernels: two CTAs of 512 threads per SM, or -- with the coarse copies, which
// double the staged image -- one CTA of 1024
#ifndef FN_BEAM_THREADS
#define FN_BEAM_THREADS 512
#endif
constexpr int kBeamThreads = FN_BEAM_THREADS;                     // threads per CTA of the beam kernels (two CTAs per SM)
template <bool kCoarse> struct FastShape { static constexpr int kThreads = kCoarse ? 1024 : kBeamThreads, kCtas = kCoarse ? 1 : 2; };
struct FastWarp {
    uint32_t slot;               // shared address of the warp's FastSlot
    uint32_t tab;                // shared address of the beam table
    uint32_t tab_last;           // ... and of its last entry
    uint32_t queue;              // shared address of the warp's queue
    uint32_t map_base;           // shared address of the staged map (for the deferred beams)
    unsigned qn;                 // entries queued (warp-uniform)
    unsigned rays;               // beams cast by this warp (warp-uniform)
};
__host__ __device__ inline void fast_chunking(int B, int* chunk_rounds, int* nchunk) {
    const int rounds = (B + 31) >> 5;
    *nchunk = (rounds + 3) >> 2;                                   // about 4 rounds = 128 beams per task
    *chunk_rounds = (rounds + *nchunk - 1) / *nchunk;
}
// magic = ceil(2^32 / d) gives t / d = umulhi(t, magic) exactly for all t < t_max when t_max * d <= 2^32; else 0 (divide)
inline unsigned fast_magic(unsigned long long d, unsigned long long t_max) {
    if (d <= 1 || t_max * d > (1ull << 32)) return 0u;
    return (unsigned)(((1ull << 32) + d - 1) / d);
}
__device__ __forceinline__ float* ring_row_of(const BeamArgs& a, const unsigned long long ring_head, const unsigned e) {
    if (!a.ring_obs) return nullptr;
    unsigned long long slot = ring_head + (unsigned long long)e;   // both < ring_cap
    if (slot >= a.ring_cap) slot -= a.ring_cap;
    return a.ring_obs + slot * (unsigned long long)a.ring_row;
}
template <int kWarps>
__device__ __forceinline__ FastWarp fast_warp(const BeamArgs& a, FastShared<kWarps>* fs, const double2* s_tab, const uint32_t map_base) {
    const unsigned wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
    FastWarp w;
    w.slot = opaque((uint32_t)__cvta_generic_to_shared(&fs->slot[wib]));
    w.tab = opaque((uint32_t)__cvta_generic_to_shared(s_tab));
    w.tab_last = opaque(w.tab + 16u * ((unsigned)a.robot.B - 1u));
    w.queue = opaque((uint32_t)__cvta_generic_to_shared(fs->queue[wib]));
    w.map_base = map_base; w.qn = 0u; w.rays = 0u;
    if (lane < 2) {                                                // the constants of the two copies
        FastAxis* ax = &fs->slot[wib].ax[lane];
        const unsigned rowBytes = (unsigned)(a.map.H + 2 * kLineGuard) * (unsigned)(a.map.strideR << 2);
        const uint32_t S = (uint32_t)(lane ? a.map.strideC : a.map.strideR) << 5;
        ax->Sd = (double)S; ax->base = map_base - a.exp_off + (lane ? rowBytes : 0u); ax->half_S = S >> 1;
        ax->inv_magic = lane ? a.inv_magicC : a.inv_magicR; ax->S = S;
        // the coarse copies follow the fine ones (padded to 16 bytes) when they are staged
        const unsigned fineBytes = ((rowBytes + (unsigned)(a.map.W + 2 * kLineGuard) * (unsigned)(a.map.strideC << 2)) + 15u) & ~15u;
        ax->base_c = map_base - a.exp_off + fineBytes + (lane ? (unsigned)coarse_words(a.map.H, a.map.strideR) * 4u : 0u);
        ax->par = 0u;
    }
    __syncwarp();
    return w;
}
// casts n (<= 32) queued beams, one per lane (queue = shared address of the first of them)
__device__ __noinline__ void fast_drain(const BeamArgs& a, const uint32_t queue, const unsigned n, const uint32_t map_base,
                                        const uint32_t tab, const unsigned long long ring_head) {
    const unsigned lane = threadIdx.x & 31;
    if (lane < n) {
        BeamMap<SmemSpace> bm;
        const int mapWords = (a.map.H + 2 * kLineGuard) * a.map.strideR + (a.map.W + 2 * kLineGuard) * a.map.strideC;
        bm.base = map_base; bm.H = a.map.H; bm.W = a.map.W; bm.stride4R = a.map.strideR << 2; bm.stride4C = a.map.strideC << 2;
        bm.rowBytes = (unsigned)(a.map.H + 2 * kLineGuard) * (unsigned)(a.map.strideR << 2);
        bm.mapBytes = (unsigned)mapWords * 4u; bm.oob = nullptr;
        const unsigned o = SmemSpace::ld(queue + 4u * lane);
        const unsigned B = (unsigned)a.robot.B;
        const unsigned e = o / B, j = o - e * B;
        const BeamPose* pose = a.poses + e;
        // cast_beam: the line-pointer form of the traversal (bit-identical to cast_beam_fast, tested), which sends
        // beams of M >= 30.5 to the word walk itself -- so a beam gets the same range whichever kernel defers it
        int hit;
        uint32_t words = 0;
        const float r = cast_beam<SmemSpace, false>(bm, pose, lds_d2(tab + 16u * j), a.robot.T, a.map.rho, a.robot.rmax, &hit, words);
        a.out_ranges[e * a.out_stride + a.out_off + j] = r;
        float* ring_row = ring_row_of(a, ring_head, e);
        if (ring_row) ring_row[a.out_off + j] = r;
    }
    __syncwarp();
}
// the rounds of a task: 32 beams each, one per lane (the env's slot is staged)
template <bool kCoarse, bool kRing>
__device__ __forceinline__ void fast_rounds(const BeamArgs& a, FastWarp& w, const int state, const unsigned e,
                                            const unsigned jb0, const unsigned jb1, const unsigned long long ring_head) {
    const unsigned lane = threadIdx.x & 31;
    const unsigned B = (unsigned)a.robot.B;
    unsigned j = jb0 + lane;
    float* po = a.out_ranges + (e * a.out_stride + a.out_off + j); // n_envs * row length < 2^31 (fn_sim_create)
    float* pr = kRing ? ring_row_of(a, ring_head, e) + (a.out_off + j) : nullptr;
    uint32_t tj = w.tab + 16u * j;
#pragma unroll 1
    for (unsigned jb = jb0; jb < jb1; jb += 32u, j += 32u, po += 32, pr += 32, tj += 512u) {
        bool near = false;
        float r = 0.0f;
        if (state == 0) r = cast_beam_fast<kCoarse>(w.slot, min(tj, w.tab_last), a.robot.T, a.half_T, a.map.rho, a.robot.rmax, near);
        const bool act = j < B;
        const unsigned nm = __ballot_sync(0xffffffffu, near && act);
        if (act && !near) {
            *po = r;
            if (kRing) *pr = r;
        }
        if (nm) {                                                  // (rare: the warp's beams cross an axis)
            if (near && act) asm volatile("st.shared.u32 [%0], %1;" ::"r"(w.queue + 4u * (w.qn + __popc(nm & ((1u << lane) - 1u)))), "r"(e * B + j) : "memory");
            w.qn += __popc(nm);
            __syncwarp();
            if (w.qn >= 32u) { w.qn -= 32u; fast_drain(a, w.queue + 4u * w.qn, 32u, w.map_base, w.tab, ring_head); }
        }
    }
}
// a near-axis beam cast on the spot (all lanes call; `mine` = this lane has one): fast_drain's cast for one beam
template <bool kCg>
__device__ __noinline__ float fast_near_beam(const BeamArgs& a, const FastWarp& w, const BeamPose* pose, const unsigned j, const bool mine, float r) {
    if (mine) {
        BeamMap<SmemSpace> bm;
        const int mapWords = (a.map.H + 2 * kLineGuard) * a.map.strideR + (a.map.W + 2 * kLineGuard) * a.map.strideC;
        bm.base = w.map_base; bm.H = a.map.H; bm.W = a.map.W; bm.stride4R = a.map.strideR << 2; bm.stride4C = a.map.strideC << 2;
        bm.rowBytes = (unsigned)(a.map.H + 2 * kLineGuard) * (unsigned)(a.map.strideR << 2);
        bm.mapBytes = (unsigned)mapWords * 4u; bm.oob = nullptr;
        BeamPose lp;
        const uint4* src = reinterpret_cast<const uint4*>(pose);
#pragma unroll
        for (int k = 0; k < (int)(sizeof(BeamPose) / 16); ++k) reinterpret_cast<uint4*>(&lp)[k] = kCg ? __ldcg(src + k) : src[k];
        int hit;
        uint32_t words = 0;
        r = cast_beam<SmemSpace, false>(bm, &lp, lds_d2(w.tab + 16u * j), a.robot.T, a.map.rho, a.robot.rmax, &hit, words);
    }
    __syncwarp();
    return r;
}
// One round of env e (beams jb0 .. jb0 + 31) with the results HELD BACK in registers, for a kernel that may cast
// before it may write (prepared_reset_kernel): fast_store_held stores them.  Near-axis beams are cast on the spot by
// cast_beam (the call fast_drain makes for them) instead of being queued: that kernel's warps cast a round or two
// each, so a queue would be drained one or two beams at a time, a second pass as long as the round.
// kCg: the pose is read past L1 (written by a kernel that may still be running).
struct HeldRound {
    float r;
    unsigned e, j;
    bool store;
};
template <bool kCg>
__device__ __forceinline__ HeldRound fast_round_held(const BeamArgs& a, FastWarp& w, const BeamPose* pose, const unsigned e, const unsigned jb0) {
    const unsigned lane = threadIdx.x & 31;
    const unsigned B = (unsigned)a.robot.B;
    __syncwarp();
    if (lane < 3) {
        const uint4* src = reinterpret_cast<const uint4*>(reinterpret_cast<const char*>(pose) + 32u * lane);
        const uint4 v = kCg ? __ldcg(src) : *src;
        asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(w.slot + ((0x401000u >> (8u * lane)) & 0xffu)),
                     "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");     // slot offsets 0, 16, 64 (fast_chunk)
    }
    const int state = kCg ? __ldcg(&pose->state) : pose->state;
    __syncwarp();
    w.rays += min(B, jb0 + 32u) - jb0;
    HeldRound h;
    h.e = e; h.j = jb0 + lane; h.r = 0.0f;
    h.store = h.j < B;
    bool near = false;
    if (state == 0) h.r = cast_beam_fast<false>(w.slot, min(w.tab + 16u * h.j, w.tab_last), a.robot.T, a.half_T, a.map.rho, a.robot.rmax, near);
    if (__any_sync(0xffffffffu, near && h.store)) h.r = fast_near_beam<kCg>(a, w, pose, h.j, near && h.store, h.r);
    return h;
}
__device__ __forceinline__ void fast_store_held(const BeamArgs& a, const HeldRound& h, const unsigned long long ring_head) {
    if (h.store) {
        a.out_ranges[h.e * a.out_stride + a.out_off + h.j] = h.r;
        if (a.ring_obs) ring_row_of(a, ring_head, h.e)[a.out_off + h.j] = h.r;
    }
}
// one task: beams [jb0, jb1) of env e, jb0 a multiple of 32 (pose = the env's sensing pose, possibly a shared-memory copy)
template <bool kCoarse>
__device__ __forceinline__ void fast_chunk(const BeamArgs& a, FastWarp& w, const BeamPose* pose, const unsigned e,
                                           const unsigned jb0, const unsigned jb1, const unsigned long long ring_head) {
    const unsigned lane = threadIdx.x & 31;
    const unsigned B = (unsigned)a.robot.B;
    // the env's part of the warp's slot: heading, (h, ouMS) of both axes
    __syncwarp();
    if (lane < 3) {
        const uint4 v = *reinterpret_cast<const uint4*>(reinterpret_cast<const char*>(pose) + 32u * lane);
        asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(w.slot + ((0x401000u >> (8u * lane)) & 0xffu)),
                     "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");     // slot offsets 0, 16, 64
        if (kCoarse && lane) asm volatile("st.shared.u32 [%0], %1;" ::"r"(w.slot + (lane == 1 ? 60u : 108u)), "r"(pose->line_par[lane - 1]) : "memory");
    }
    const int state = pose->state;
    __syncwarp();
    w.rays += jb1 - jb0;
    if (a.ring_obs) fast_rounds<kCoarse, true>(a, w, state, e, jb0, jb1, ring_head);    // (two copies of the round loop: a
    else fast_rounds<kCoarse, false>(a, w, state, e, jb0, jb1, ring_head);              //  predicated-off ring store still issues)
}

// words of the staged image with the coarse copies: fine copies (padded to 16 bytes), then the coarse ones
__host__ __device__ inline int staged_words_coarse(const MapDev& m) {
    const int fine = (m.H + 2 * kLineGuard) * m.strideR + (m.W + 2 * kLineGuard) * m.strideC;
    return ((fine + 3) & ~3) + (int)((coarse_words(m.H, m.strideR) + coarse_words(m.W, m.strideC) + 3) / 4 * 4);
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
    // (try_wait gives up after a system-dependent time and is simply asked again: the copies were issued by this CTA
    // from addresses the host checked, so they complete -- or fault on their own; a bound on the polls could only
    // misfire under a debugger or a time-sliced context, and there is nothing sensible to do without the map)
    uint32_t done = 0;
    while (!done)
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(mb) : "memory");
}

// The warps of the (persistent) grid take their tasks in two parts.  Beams differ in length by an order of
// magnitude, and a purely static split leaves ~15 % of the SM time idle at the end of the launch.  So: the
// first 3/4 of each warp's share is static (round r -> task warp0 + r * nwarps, no atomics), the rest is
// handed out dynamically, one atomic per warp task, fetched one task ahead so that its latency is hidden.
// (has_static = false: a warp that arrives late -- fn_step_split.cuh -- takes pool tasks only)
struct TaskFeed {
    unsigned ntasks, warp0, nwarps, static_rounds, dyn_base, round, task;
    bool dynamic;
    unsigned* counter;
    __device__ __forceinline__ TaskFeed(const unsigned ntasks_, const unsigned warp0_, const unsigned nwarps_,
                                        const bool has_static, unsigned* counter_)
        : ntasks(ntasks_), warp0(warp0_), nwarps(nwarps_), counter(counter_) {
        static_rounds = max(1u, ((ntasks / nwarps) * 3u) >> 2);
        dyn_base = static_rounds * nwarps;
        dynamic = dyn_base < ntasks;                               // (short launches are static only)
        round = 0;
        task = warp0;
        if (!has_static) {
            round = static_rounds;
            task = ntasks;
            if (dynamic && (threadIdx.x & 31) == 0) task = dyn_base + atomicAdd(counter, 1u);
            task = __shfl_sync(0xffffffffu, task, 0);
        }
    }
    __device__ __forceinline__ bool valid() const { return task < ntasks; }
    // issue the fetch of the task after this one (call before working on `task`) ...
    __device__ __forceinline__ unsigned prefetch() {
        unsigned next = ntasks;
        ++round;
        if (round < static_rounds) next = warp0 + round * nwarps;
        else if (dynamic && (threadIdx.x & 31) == 0) next = dyn_base + atomicAdd(counter, 1u);
        return next;
    }
    // ... and move on to it (after the work)
    __device__ __forceinline__ void advance(const unsigned next) { task = __shfl_sync(0xffffffffu, next, 0); }
};

// Instrumented / L2-path kernels: a task = 32 consecutive (env, beam) pairs: adjacent lanes = adjacent beams of
// one env, so a warp's loads mostly hit the same or neighbouring words and its lanes run similar trip counts.
template <class MS, bool kAux>
__device__ __forceinline__ void run_beam_tasks(const BeamArgs& a, const BeamMap<MS>& bm,
                                               const double2* s_tab, const int* list, const int n_env, const unsigned total,
                                               const unsigned long long ring_head,     // slot of env 0's pending ring row
                                               const unsigned warp0, const unsigned nwarps,  // this warp's place among the
                                               const bool has_static = true) {         // warps that share the static part
    const int B = a.robot.B;
    const int lane = threadIdx.x & 31;
    uint32_t words = 0, rays = 0;
    const unsigned long long invB = ~0ull / (unsigned long long)B + 1ull;     // floor(2^64 / B) + 1
    TaskFeed feed((total + 31u) >> 5, warp0, nwarps, has_static, a.task_counter);
    while (feed.valid()) {
        const unsigned next = feed.prefetch();
        // (listed env, beam) of this lane's element idx = 32 task + lane
        const unsigned idx = (feed.task << 5) + lane;
        const unsigned le = B > 1 ? (unsigned)__umul64hi((unsigned long long)idx, invB) : idx;   // idx / B, exact for idx < 2^32 (B = 1: invB wraps to 0)
        const unsigned j = idx - le * (unsigned)B;
        if (le < (unsigned)n_env) {
            const unsigned e = list ? (unsigned)list[le] : le;
            beam_element<MS, kAux>(a, bm, s_tab, a.poses + e, e, j, ring_head, words);
            ++rays;
        }
        feed.advance(next);
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

__device__ __forceinline__ void fast_finish(const BeamArgs& a, FastWarp& w, const unsigned long long ring_head) {
    if (w.qn) fast_drain(a, w.queue, w.qn, w.map_base, w.tab, ring_head);
    if ((threadIdx.x & 31) == 0 && w.rays) atomicAdd(&a.counters[kRays], (unsigned long long)w.rays);
}
// The envs' beams as warp tasks, handed out in order by one atomic counter (fetched one task ahead, so that its
// latency is hidden; a warp's first task is its own index).  Two sizes: the first 24/32 of the envs go out in chunks
// of chunk_rounds x 32 beams -- what depends on the env is amortised over the chunk -- and the rest in single
// rounds of 32 beams, so that the launch ends within one round's time on every SM (beams differ in length by an
// order of magnitude; a static split of such chunks left 13 % of the SM time idle).  Small launches (fewer than
// eight rounds per warp) use single rounds only.
// (has_static = false: a warp that arrives late -- fn_step_split.cuh -- has no task of its own)
template <bool kCoarse>
__device__ __forceinline__ void run_fast_tasks(const BeamArgs& a, FastWarp& w, const int* list, const int n_env,
                                               const unsigned long long ring_head, const unsigned warp0,
                                               const unsigned nwarps, const bool has_static = true) {
    const unsigned B = (unsigned)a.robot.B, rounds = (B + 31u) >> 5;
    const unsigned nchunk = (unsigned)a.nchunk, cbeams = (unsigned)a.chunk_rounds << 5;
    const unsigned nA = (unsigned)n_env * rounds >= 8u * nwarps ? ((unsigned)n_env * 24u) >> 5 : 0u;   // envs cast in chunks
    const unsigned ntA = nA * nchunk, nt = ntA + ((unsigned)n_env - nA) * rounds;
    const unsigned lane = threadIdx.x & 31;
    unsigned t = warp0;
    if (!has_static) {
        if (lane == 0) t = nwarps + atomicAdd(a.task_counter, 1u);
        t = __shfl_sync(0xffffffffu, t, 0);
    }
    while (t < nt) {
        unsigned next = 0u;
        if (lane == 0) next = nwarps + atomicAdd(a.task_counter, 1u);
        unsigned le, jb0, jb1;
        if (t < ntA) {
            le = a.inv_nchunk ? __umulhi(t, a.inv_nchunk) : t / nchunk;               // (exact: fast_magic)
            jb0 = (t - le * nchunk) * cbeams;
            jb1 = jb0 + cbeams;
        } else {
            const unsigned u = t - ntA;
            const unsigned lb = a.inv_rounds ? __umulhi(u, a.inv_rounds) : u / rounds;
            le = nA + lb;
            jb0 = (u - lb * rounds) << 5;
            jb1 = jb0 + 32u;
        }
        const unsigned e = list ? (unsigned)list[le] : le;
        fast_chunk<kCoarse>(a, w, a.poses + e, e, jb0, min(B, jb1), ring_head);
        t = __shfl_sync(0xffffffffu, next, 0);
    }
    fast_finish(a, w, ring_head);
}

// Persistent kernel (grid = SMs x resident CTAs).  kSmem: each CTA stages both packed copies of the map
// and the beam table in shared memory -- constants, so this happens BEFORE the dependency wait, under
// the env-step / reset kernel that precedes it in the stream.
// kAux = instrumented variant: hit-cell output, map-word counter.
// kCoarse (production kernel only): the coarse copies are staged too and the hot loop walks them.
template <bool kSmem, bool kAux, bool kCoarse = false>
__global__ void __launch_bounds__(FastShape<kCoarse>::kThreads, FastShape<kCoarse>::kCtas) beam_kernel(const __grid_constant__ BeamArgs a) {
    static_assert(!kCoarse || (kSmem && !kAux), "the coarse level belongs to the production kernel");
    extern __shared__ __align__(16) uint8_t smem_raw[];
    const int B = a.robot.B;
    constexpr bool stage = kSmem;
    constexpr bool fast = kSmem && !kAux;
    const int mapWords = (a.map.H + 2 * kLineGuard) * a.map.strideR + (a.map.W + 2 * kLineGuard) * a.map.strideC;
    double2* s_tab = reinterpret_cast<double2*>(smem_raw);
    uint32_t* s_map = reinterpret_cast<uint32_t*>(smem_raw + (size_t)B * sizeof(double2));
    __shared__ __align__(8) unsigned long long s_mbar;
    __shared__ __align__(16) typename std::conditional<fast, FastShared<FastShape<kCoarse>::kThreads / 32>, int>::type s_fast;
    stage_beam_constants(a, s_tab, s_map, kCoarse ? staged_words_coarse(a.map) : mapWords, stage, &s_mbar);
    __syncthreads();
    griddep_wait();                                                // poses / list / count come from the previous kernel
    griddep_launch_dependents();
    if (a.flip_par_dev && blockIdx.x == 0 && threadIdx.x == 0) {
        const int p = *a.flip_par_dev;
        a.done_count[p ^ 1] = 0;
        *a.flip_par_dev = p ^ 1;
    }
    const int* list = a.list;
    const int* count_dev = a.count_dev;
    if (a.list_par_dev) { const int q = *a.list_par_dev ^ 1; list += (size_t)q * a.n_all; count_dev += q; }
    const int n_env = count_dev ? *count_dev : a.n_all;
    const unsigned total = (unsigned)n_env * (unsigned)B;
    const unsigned long long ring_head = a.ring_obs ? *a.ring_head : 0ull;
    const unsigned warp0 = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const unsigned nwarps = gridDim.x * (blockDim.x >> 5);

    const unsigned rowBytes = (unsigned)(a.map.H + 2 * kLineGuard) * (unsigned)(a.map.strideR << 2);
    if constexpr (fast) {
        FastWarp w = fast_warp(a, &s_fast, s_tab, (uint32_t)__cvta_generic_to_shared(s_map));
        run_fast_tasks<kCoarse>(a, w, list, n_env, ring_head, warp0, nwarps);
    } else if (stage) {
        BeamMap<SmemSpace> bm;
        bm.base = (uint32_t)__cvta_generic_to_shared(s_map);
        bm.H = a.map.H; bm.W = a.map.W; bm.stride4R = a.map.strideR << 2; bm.stride4C = a.map.strideC << 2;
        bm.rowBytes = rowBytes; bm.mapBytes = (unsigned)mapWords * 4u; bm.oob = a.counters + kOobLoads;
        run_beam_tasks<SmemSpace, kAux>(a, bm, s_tab, list, n_env, total, ring_head, warp0, nwarps);
    } else {
        BeamMap<GlobalSpace> bm;
        bm.base = (unsigned long long)__cvta_generic_to_global(a.map.row);
        bm.H = a.map.H; bm.W = a.map.W; bm.stride4R = a.map.strideR << 2; bm.stride4C = a.map.strideC << 2;
        bm.rowBytes = rowBytes; bm.mapBytes = (unsigned)mapWords * 4u; bm.oob = a.counters + kOobLoads;
        run_beam_tasks<GlobalSpace, kAux>(a, bm, s_tab, list, n_env, total, ring_head, warp0, nwarps);
    }
}

}  // namespace fn
