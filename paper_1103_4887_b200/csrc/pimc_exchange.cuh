// Deterministic scalar all-reduce between the co-resident CTAs of one chain: the grid-wide sum that every parameter
// move needs (row A4 of SURVEY.md §8(a); "block sums ... a second kernel sums them and decides").
//
// Round 1 ran a flat all-gather: every CTA published its block sum in one 128-byte mailbox line and all G CTAs polled
// all G lines (G x G polls, 148 readers per line): ~1900 cycles until the last packet had been seen everywhere, plus two
// block sums with a barrier each (profiles/r01_v8_final.md: `barrier` + `long_scoreboard` on top of the A4 stalls).
// This file holds the round-2 exchange, a two-hop butterfly run by ONE warp per CTA:
//   hop 1 (row)   : the CTAs are laid out as rows x cols.  Every WARP publishes its own partial (no block barrier before
//                   the store) as a 16-byte tagged packet in its CTA's line A; the exchange warp of every CTA of the row
//                   polls the cols x NW packets of its row (<= 4 packets per lane, all loads in flight together), sums
//                   them in a fixed order (lane-serial, then xor tree) -- every CTA of the row gets the same bits;
//   hop 2 (column): lane 0 publishes the row sum in line B; the exchange warp polls the `rows` row sums of its column
//                   (one packet per lane), same xor tree in every CTA => the total is bit-identical grid-wide, so all
//                   CTAs take the same accept decision without a broadcast (fixed order, reproducible).
// A line now has <= cols (or rows) reader CTAs instead of G.  Packets are {payload32, tag32} pairs as in
// pimc_tile_kernel.cuh: relaxed 8/16-byte accesses, no fence, no separate flag; the tag is the all-reduce epoch, and
// two mailbox buffers alternate (a CTA can be at most one all-reduce ahead of any other, see xchg_warp_2d).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace pimc {

constexpr int kXchgMaxCtas = 256;          // co-resident CTAs of a launch (one per SM)
constexpr int kXchgWarps = 8;              // packets in line A: one per warp of a 256-thread CTA
constexpr int kXchgLineWords = 16;         // 128 bytes
constexpr int kXchgCtaWords = 2 * kXchgLineWords;                 // line A (warp partials) + line B (row sum)
constexpr size_t kXchgWords = (size_t)2 * kXchgMaxCtas * kXchgCtaWords;   // two alternating buffers
constexpr unsigned long long kXchgSpinLimit = 20ull * 1000 * 1000;

__device__ __forceinline__ void xchg_store(unsigned long long* p, double v, uint32_t tag) {
    const unsigned long long bits = (unsigned long long)__double_as_longlong(v), t = (unsigned long long)tag << 32;
    asm volatile("st.relaxed.gpu.global.v2.u64 [%0], {%1, %2};" ::"l"(p), "l"(t | (bits & 0xFFFFFFFFull)), "l"(t | (bits >> 32)) : "memory");
}
__device__ __forceinline__ bool xchg_try(const unsigned long long* p, uint32_t tag, double& v) {
    unsigned long long a, b;
    asm volatile("ld.relaxed.gpu.global.v2.u64 {%0, %1}, [%2];" : "=l"(a), "=l"(b) : "l"(p) : "memory");
    v = __longlong_as_double((long long)((b << 32) | (a & 0xFFFFFFFFull)));
    return (uint32_t)(a >> 32) == tag && (uint32_t)(b >> 32) == tag;
}

// The same load under a predicate INSIDE the asm statement: a C++ `if` around an asm block becomes a branch, and the loads of a
// multi-packet poll would then wait for one another (one L2 round trip each) instead of being in flight together.
__device__ __forceinline__ bool xchg_try_if(bool want, const unsigned long long* p, uint32_t tag, double& v) {
    unsigned long long a = 0, b = 0;
    asm volatile("{\n\t.reg .pred q;\n\tsetp.ne.u32 q, %3, 0;\n\t@q ld.relaxed.gpu.global.v2.u64 {%0, %1}, [%2];\n\t}"
                 : "+l"(a), "+l"(b) : "l"(p), "r"((unsigned)want) : "memory");
    v = __longlong_as_double((long long)((b << 32) | (a & 0xFFFFFFFFull)));
    return want && (uint32_t)(a >> 32) == tag && (uint32_t)(b >> 32) == tag;
}

struct XchgGeom {
    int G, b, cols, rows, row, col, n_mem;      // n_mem = CTAs in my row
};
__host__ __device__ inline int xchg_cols(int G, int nw) {
    int c = 1;
    while (c * c < G) ++c;                      // ceil(sqrt(G)): rows <= cols
    const int cap = 128 / nw;                   // <= 4 packets per lane in hop 1
    return c < cap ? c : cap;
}
__device__ __forceinline__ XchgGeom xchg_geom(int G, int b, int nw) {
    XchgGeom g;
    g.G = G; g.b = b; g.cols = xchg_cols(G, nw); g.rows = (G + g.cols - 1) / g.cols;
    g.row = b / g.cols; g.col = b % g.cols;
    g.n_mem = min(g.cols, G - g.row * g.cols);
    return g;
}

__device__ __forceinline__ unsigned long long* xchg_line(unsigned long long* mbox, int buf, int cta, int which) {
    return mbox + ((size_t)buf * kXchgMaxCtas + (size_t)cta) * kXchgCtaWords + (size_t)which * kXchgLineWords;
}

// Called by lane 0 of every warp of the CTA with that warp's partial (any time after the previous all-reduce was consumed).
__device__ __forceinline__ void xchg_publish_warp(unsigned long long* mbox, int buf, int cta, int warp, double v, uint32_t tag) {
    xchg_store(xchg_line(mbox, buf, cta, 0) + 2 * warp, v, tag);
}

__device__ __forceinline__ double xchg_xor_tree(double v) {
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, off);
    return v;
}

// Flat gather by ONE warp: packet j (16 bytes at base + j * stride_words) of every CTA j < G <= 256, own value passed in
// (not re-read).  Lane i takes packets i, i + 32, ...: all of a lane's loads are in flight together; the sum is lane-serial in
// index order, then a fixed xor tree -- the same bits in every CTA.
__device__ __forceinline__ double xchg_gather_warp(const unsigned long long* base, int stride_words, int G, int b, double own,
                                                   uint32_t tag, int* fault) {
    const int lane = threadIdx.x & 31;
    double v[8];
    unsigned pend = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const int j = lane + 32 * k;
        v[k] = j == b ? own : 0.0;
        if (j < G && j != b) pend |= 1u << k;
    }
    unsigned long long spins = 0;
    while (pend) {
        double t[8];
        bool ok[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) ok[k] = xchg_try_if(pend >> k & 1u, base + (size_t)(lane + 32 * k) * stride_words, tag, t[k]);
#pragma unroll
        for (int k = 0; k < 8; ++k) if (ok[k]) { v[k] = t[k]; pend &= ~(1u << k); }
        if (++spins > kXchgSpinLimit) { atomicExch(fault, 1); break; }
        if ((spins & 0xFFFFull) == 0 && *reinterpret_cast<volatile int*>(fault) != 0) break;
    }
    __syncwarp();
    return xchg_xor_tree(((v[0] + v[1]) + (v[2] + v[3])) + ((v[4] + v[5]) + (v[6] + v[7])));
}

// ---- order-independent all-reduce: fixed-point integer accumulation in L2 ------------------------------------------------------
// Each CTA converts its partial to a 120-bit offset-binary fixed-point number (64 fractional bits; |partial| < 2^55, anything
// else -- NaN, inf, absurdly large -- is counted as "bad" and makes the total NaN, i.e. the move is rejected),
// splits it into three 40-bit limbs and adds each limb to its own 64-bit accumulator word with a fire-and-forget
// red.global.add: integer addition is associative, so the total does not depend on the arrival order (run-to-run
// bit-reproducible, reading G19) and every CTA reads the SAME words, hence the same decision, with no gather and no second
// block sum.  Word layout: bits 0..47 limb sum (40 bits + headroom for 256 CTAs), bits 48..63 number of contributions so
// far (mod 2^16); word 3 counts bad contributions (same count field).  The words are never zeroed: tile 0 of the chain adds
// its limb MINUS the limb field left by the previous use of the buffer (which every CTA knows: it is what they all read), and
// the count field just keeps running, so a stale word can never look complete.  Two buffers alternate, as above.
struct XfixState {
    unsigned long long last[2][4];     // the completed words of each buffer as everybody last read them
};
constexpr int kXfixLineWords = 16;     // one 128-byte line per (chain, buffer)
constexpr unsigned long long kXfixLimbMask = (1ull << 48) - 1ull;

__device__ __forceinline__ void xfix_red_add(unsigned long long* p, unsigned long long v) {
    asm volatile("red.relaxed.gpu.global.add.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
// partial -> three 40-bit limbs of trunc(partial * 2^64) + 2^119; returns false if the partial is not representable
__device__ __forceinline__ bool xfix_split(double v, unsigned long long limb[3]) {
    const unsigned long long bits = (unsigned long long)__double_as_longlong(v);
    const int e = (int)((bits >> 52) & 0x7FFull);
    const bool ok = e < 1023 + 55;                                   // |v| < 2^55 and finite
    const unsigned long long m = e ? ((bits & 0xFFFFFFFFFFFFFull) | (1ull << 52)) : 0ull;   // subnormals are far below 2^-64
    const int s = e - 1011;                                          // v = m 2^(e-1075)  =>  v 2^64 = m 2^s, s <= 66
    unsigned __int128 mag = 0;
    if (ok) {
        if (s >= 0) mag = (unsigned __int128)m << s;
        else if (s > -64) mag = (unsigned __int128)(m >> -s);
    }
    const __int128 n = (bits >> 63) ? -(__int128)mag : (__int128)mag;
    const unsigned __int128 u = (unsigned __int128)(n + ((__int128)1 << 119));
    constexpr unsigned long long k40 = (1ull << 40) - 1ull;
    limb[0] = (unsigned long long)u & k40;
    limb[1] = (unsigned long long)(u >> 40) & k40;
    limb[2] = (unsigned long long)(u >> 80) & k40;
    return ok;
}
// limb sums of G contributions -> double (one rounding of the exact integer total)
__device__ __forceinline__ double xfix_join(const unsigned long long L[3], int G) {
    const unsigned __int128 u = (unsigned __int128)L[0] + ((unsigned __int128)L[1] << 40) + ((unsigned __int128)L[2] << 80);
    const __int128 n = (__int128)u - ((__int128)G << 119);
    const bool neg = n < 0;
    const unsigned __int128 mag = neg ? (unsigned __int128)(-n) : (unsigned __int128)n;
    const unsigned long long hi = (unsigned long long)(mag >> 64), lo = (unsigned long long)mag;
    double d;
    if (hi == 0ull) d = __ull2double_rn(lo) * 0x1p-64;
    else {
        const int sh = __clzll((long long)hi);                        // 0..63
        const unsigned long long top = sh ? ((hi << sh) | (lo >> (64 - sh))) : hi;
        d = __ull2double_rn(top) * __longlong_as_double((long long)(1023 - sh) << 52);     // top 2^(64-sh) 2^-64
    }
    return neg ? -d : d;
}
// The whole all-reduce, run by ONE thread per CTA.  acc: this chain's accumulator lines [2 buffers][kXfixLineWords]; first =
// this CTA is tile 0 of the chain; count = all-reduces this chain has finished (buffer = count & 1).
__device__ __forceinline__ double xfix_allreduce(unsigned long long* acc, XfixState& st, int G, bool first, unsigned long long count,
                                                 double v, int* fault) {
    const int buf = (int)(count & 1ull);
    unsigned long long* w = acc + (size_t)buf * kXfixLineWords;
    unsigned long long limb[3];
    const bool ok = xfix_split(v, limb);
    const unsigned long long one = 1ull << 48;
#pragma unroll
    for (int k = 0; k < 3; ++k) xfix_red_add(w + k, limb[k] + one - (first ? (st.last[buf][k] & kXfixLimbMask) : 0ull));
    xfix_red_add(w + 3, (ok ? 0ull : 1ull) + one - (first ? (st.last[buf][3] & kXfixLimbMask) : 0ull));
    const unsigned long long want = ((st.last[buf][0] >> 48) + (unsigned long long)G) & 0xFFFFull;
    unsigned long long a, b, c, d, spins = 0;
    for (;;) {
        asm volatile("ld.relaxed.gpu.global.v2.u64 {%0, %1}, [%2];" : "=l"(a), "=l"(b) : "l"(w) : "memory");
        asm volatile("ld.relaxed.gpu.global.v2.u64 {%0, %1}, [%2];" : "=l"(c), "=l"(d) : "l"(w + 2) : "memory");
        if ((a >> 48) == want && (b >> 48) == want && (c >> 48) == want && (d >> 48) == want) break;
        if (++spins > kXchgSpinLimit) { atomicExch(fault, 1); break; }
        if ((spins & 0xFFFFull) == 0 && *reinterpret_cast<volatile int*>(fault) != 0) break;
    }
    st.last[buf][0] = a; st.last[buf][1] = b; st.last[buf][2] = c; st.last[buf][3] = d;
    const unsigned long long L[3] = {a & kXfixLimbMask, b & kXfixLimbMask, c & kXfixLimbMask};
    const double tot = xfix_join(L, G);
    return (d & kXfixLimbMask) ? __longlong_as_double(0x7FF8000000000000ll) : tot;
}
// At kernel start (the previous launch has completed, the words are quiescent): read both buffers.
__device__ __forceinline__ void xfix_begin(const unsigned long long* acc, XfixState& st) {
#pragma unroll
    for (int buf = 0; buf < 2; ++buf)
#pragma unroll
        for (int k = 0; k < 4; ++k) st.last[buf][k] = __ldcg(acc + (size_t)buf * kXfixLineWords + k);
}

// The two hops, run by one full warp.  mbox: this chain's mailbox (CTA index = tile index b); nw = warps per CTA that
// publish; tag = epoch + 1, buf = epoch & 1.  Returns the grid-wide sum in every lane.
// Why two buffers suffice: a CTA finishes all-reduce k only after every CTA has published its hop-1 packets of k, i.e.
// after every CTA has finished READING all-reduce k-1; so nobody still polls buffer (k-1)&1 = (k+1)&1 when it is rewritten.
__device__ __forceinline__ double xchg_warp_2d(unsigned long long* mbox, const XchgGeom& g, int nw, uint32_t tag, int buf, int* fault) {
    const int lane = threadIdx.x & 31;
    // ---- hop 1: the cols x nw warp partials of my row ----
    const int npk = g.cols * nw;                 // <= 128
    const int first = g.row * g.cols;
    double v[4] = {0.0, 0.0, 0.0, 0.0};
    const unsigned long long* src[4];
    unsigned pend = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int q = lane + 32 * k, m = q / nw, w = q - m * nw;
        src[k] = xchg_line(mbox, buf, first + (m < g.n_mem ? m : 0), 0) + 2 * w;
        if (q < npk && m < g.n_mem) pend |= 1u << k;
    }
    unsigned long long spins = 0;
    while (pend) {
        double t[4];
        bool ok[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) ok[k] = xchg_try_if(pend >> k & 1u, src[k], tag, t[k]);
#pragma unroll
        for (int k = 0; k < 4; ++k) if (ok[k]) { v[k] = t[k]; pend &= ~(1u << k); }
        if (++spins > kXchgSpinLimit) { atomicExch(fault, 1); break; }
        if ((spins & 0xFFFFull) == 0 && *reinterpret_cast<volatile int*>(fault) != 0) break;
    }
    __syncwarp();
    const double row_sum = xchg_xor_tree((v[0] + v[1]) + (v[2] + v[3]));
    if (g.rows == 1) return row_sum;
    // ---- hop 2: the row sums of my column ----
    if (lane == 0) xchg_store(xchg_line(mbox, buf, g.b, 1), row_sum, tag);
    double c = 0.0;
    if (lane < g.rows) {
        if (lane == g.row) c = row_sum;
        else {
            const int n_mem_r = min(g.cols, g.G - lane * g.cols);             // the last row may be short
            const unsigned long long* p = xchg_line(mbox, buf, lane * g.cols + min(g.col, n_mem_r - 1), 1);
            spins = 0;
            while (!xchg_try(p, tag, c)) {
                if (++spins > kXchgSpinLimit) { atomicExch(fault, 1); break; }
                if ((spins & 0xFFFFull) == 0 && *reinterpret_cast<volatile int*>(fault) != 0) break;
            }
        }
    }
    __syncwarp();
    return xchg_xor_tree(c);
}

}  // namespace pimc
