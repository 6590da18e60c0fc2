// tdos_main6.cuh -- main kernel "v6" of the tetrahedron-DOS hot path, the default for
// norb >= 5 with norb % 4 == 0.
//
// A BLOCK works on one item = (tile of TX x TY x TZ cubes, band, block of 8 orbitals); its warps share the tile's
// records in shared memory.  Per item:
//   stage  A1      the (TX+1)(TY+1)(TZ+1) k-points of E and W (periodic wrap, nothing materialised); the tile's
//                  lowest energy fixes the first bin pb of the item's energy span;
//   build  A2/A3   thread = (tetrahedron, band): 5 compare-exchanges carrying the corner points; the four bins
//                  i1 (first omega > E1), i2, i3, i4 (first omega >= E2, E3, E4); Eq. 15's constant sum_l b_l goes
//                  once into the step histogram S at bin i4; and -- ONCE per tetrahedron -- the parameters of its
//                  three records, one per interval of PAPER.md Eq. 12-14 (:109-195):
//                    low  [i1,i2), Eq. 12:  with s = (w-E1)/E21,  sum_l b_lm w_l = hs s^3 b_1m + hs s^4 Gq_m,
//                         hs = 4 rho, rho = (E21/E31)(E21/E41), Gq_m = 1/4 sum_{j=2,3,4} (E21/E_j1)(b_jm - b_1m);
//                    high [i3,i4), Eq. 14 (mirror image): s = (E4-w)/E43, sum_l b_lm w_l = V_m + hs s^3 b_4m + hs s^4 Gq_m
//                         with hs = -4 rho, V_m = sum_l b_lm (Eq. 14c/e's constant);
//                    mid  [i2,i3), Eq. 13: sorted energies, the reciprocals 1/E31, 1/E41, 1/E32, 1/E42, corner points;
//                  the derivative (DOS) comes from the same two vectors: d/dw = r hs (3 s^2 b + 4 s^3 Gq);
//                  energy bins are owned in chunks of 4: the records overlapping each chunk are counted per interval kind;
//   plan           the block's groups of 2 lanes are dealt out to the chunks in proportion to their cost (bisection
//                  on the load per group), so a group owns ONE chunk for the whole item and takes an equal share
//                  of that chunk's low, high and mid lists;
//   fill           every record is entered into the list of each chunk it overlaps (counting sort by (kind, chunk));
//   walk   A4-A6   the paper's "thread = energy, thread-local accumulation" (:249-253) restricted to the windows:
//                  the sums of a chunk (4 bins x 8 orbitals x {DOS, N}) stay in the registers of its group; a warp
//                  walks the low entries of its groups, then the high ones, then the mid ones, so all lanes run the
//                  same code.  Low/high: lane = 4 bins x 4 orbitals, 4-5 FMAs per orbital and bin.  Mid: lane = 2 bins
//                  x 8 orbitals, Eq. 13a-n for two bins at once (packed fp32x2), then the 4 x 8 projection;
//   flush          one vector reduction (performed in L2) of the registers into the partial histogram per group.
// Only Eq. 15 goes into the step histogram S; every fp32 sum (registers, partials, S) is a sum of non-negative
// terms bounded by N itself.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "tdos_kernels.cuh"

namespace tdos {

template <int TX, int TY, int TZ, int NWARP>
struct Cfg6 {
    static constexpr int MB = 8;
    static constexpr int PX = TX + 1, PY = TY + 1, PZ = TZ + 1;
    static constexpr int PK = PX * PY * PZ;          // k-points staged per tile
    static constexpr int NC = TX * TY * TZ;          // cubes per tile
    static constexpr int NTB = 6 * NC;               // (tetrahedron, band) per item
    static constexpr int NT = NWARP * 32;
    static constexpr int ITER = (NTB + NT - 1) / NT; // tetrahedra per thread
    static constexpr int NG = NWARP * 16;            // groups of 2 lanes
    static constexpr int NCH = 64, CH = 4;           // chunk counters, bins per chunk
    static constexpr int NCHP = (NG > 64) ? 64 : 32; // chunks per pass (fewer than groups)
    static constexpr int CAP = 8 * NTB;              // (record, chunk) entries per pass (>= 3 NTB: one chunk always fits)
    // fill: the lanes of a warp take records STRIDE apart -- neighbouring tetrahedra share their chunks, and a
    // shared-memory atomic with a returned value costs one cycle per lane on the same address
    static constexpr int STRIDE = 37;
    static_assert(PK <= 256, "corner points are 8-bit");
    static_assert(NTB <= 65535 && NTB % STRIDE != 0, "record ids are 16-bit; STRIDE must be coprime with NTB");
    static_assert(NG > NCHP, "more groups than chunks");
    static constexpr size_t a16(size_t x) { return (x + 15) / 16 * 16; }
    static constexpr size_t sz_e = a16((size_t)4 * PK), sz_w = (size_t)32 * PK;
    static constexpr size_t off_e = 0;                                    // float  [2][PK]     the tile of this item | the next one
    static constexpr size_t off_w = off_e + 2 * sz_e;                     // float  [2][PK][8]
    static constexpr size_t off_ls = off_w + 2 * sz_w;                    // float4 [NTB]     low: x0, r, hs, range
    static constexpr size_t off_lg = off_ls + (size_t)16 * NTB;           // float4 [NTB][2]  low: Gq
    static constexpr size_t off_hs = off_lg + (size_t)32 * NTB;           // float4 [NTB]     high
    static constexpr size_t off_hg = off_hs + (size_t)16 * NTB;           // float4 [NTB][2]
    static constexpr size_t off_hv = off_hg + (size_t)32 * NTB;           // float4 [NTB][2]  high: V = sum_l b_l
    static constexpr size_t off_me = off_hv + (size_t)32 * NTB;           // float4 [NTB]     mid: e1..e4
    static constexpr size_t off_mr = off_me + (size_t)16 * NTB;           // float4 [NTB]     mid: 1/e31, 1/e41, 1/e32, 1/e42
    static constexpr size_t off_rng = off_mr + (size_t)16 * NTB;          // uint4  [NTB]     ranges low, high, mid; corner points
    static constexpr size_t off_ent = off_rng + (size_t)16 * NTB;         // uint32 [CAP + 2] record | near point << 16
    static constexpr size_t off_cnt = off_ent + a16((size_t)4 * (CAP + 2));   // int [2][3][NCH] entries per (kind, chunk), by item parity
    static constexpr size_t off_off = off_cnt + (size_t)4 * 2 * 3 * NCH;  // int [3][NCH] start of the list
    static constexpr size_t off_cur = off_off + (size_t)4 * 3 * NCH;      // int [3][NCH] fill cursors
    static constexpr size_t off_gst = off_cur + (size_t)4 * 3 * NCH;      // int [NCH + 1] first group of a chunk
    static constexpr size_t off_misc = off_gst + a16((size_t)4 * (NCH + 1));
    static constexpr size_t bytes = off_misc + 128;                       // (+ a copy of omega behind it when it fits)
};

// words of sMisc: two item descriptions (by item parity) of 8 words, then the pass's chunk count
enum { M6_ITEM = 0, M6_X0, M6_Y0, M6_Z0, M6_BAND, M6_MB, M6_LMAX, M6_DESC = 8, M6_NC = 16 };

// locate_bin (tdos_kernels.cuh) on an energy array in any address space (shared-memory copy or global)
template <bool STRICT>
__device__ __forceinline__ int locate6(const float* om, int nE, float om0, float inv_dom, float x) {
    float gq = (x - om0) * inv_dom;
    gq = fminf(fmaxf(gq, 0.0f), (float)nE);
    int i = (int)gq;
    if (STRICT) {
        while (i > 0 && om[i - 1] > x) --i;
        while (i < nE && om[i] <= x) ++i;
    } else {
        while (i > 0 && om[i - 1] >= x) --i;
        while (i < nE && om[i] < x) ++i;
    }
    return i;
}

__device__ __forceinline__ void cp_async4(void* smem_dst, const void* gsrc) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// low/high walk: lane = 4 bins x 4 orbitals x {DOS, in-window N}
struct AccE6 {
    f2 D[4][2], T[4][2];
    __device__ __forceinline__ void zero() {
#pragma unroll
        for (int b = 0; b < 4; b++) { D[b][0] = D[b][1] = T[b][0] = T[b][1] = make_float2(0.f, 0.f); }
    }
};
// mid walk: lane = 2 bins x 8 orbitals x {DOS, in-window N}
struct AccM6 {
    f2 D[2][4], T[2][4];
    __device__ __forceinline__ void zero() {
#pragma unroll
        for (int b = 0; b < 2; b++)
#pragma unroll
            for (int j = 0; j < 4; j++) D[b][j] = T[b][j] = make_float2(0.f, 0.f);
    }
};

// One low (Eq. 12) or high (Eq. 14) entry for the chunk's four bins, this lane's four orbitals.
// S = {x0, r, hs, range}: s = (w - x0) r;  G, B, V: Gq, b_near, sum_l b_l at the lane's orbitals.
template <bool HIGH>
__device__ __forceinline__ void eval_edge6(AccE6& a, const float4 S, const float4 G, const float4 B, const float4 V,
                                           const f2 (&om)[2], int bin0) {
    const uint32_t rng = __float_as_uint(S.w);
    const int lo = (int)(rng & 0xffffu);
    const unsigned len = (rng >> 16) - (rng & 0xffffu);
    const f2 B01 = make_float2(B.x, B.y), B23 = make_float2(B.z, B.w);
    const f2 G01 = make_float2(G.x, G.y), G23 = make_float2(G.z, G.w);
    const f2 V01 = make_float2(V.x, V.y), V23 = make_float2(V.z, V.w);
    const f2 NX0 = dup(-S.x), R = dup(S.y), HS = dup(S.z), R4 = dup(4.0f * S.y), Q = dup(0.75f);
#pragma unroll
    for (int pr = 0; pr < 2; pr++) {
        const bool ok0 = (unsigned)(bin0 + 2 * pr - lo) < len, ok1 = (unsigned)(bin0 + 2 * pr + 1 - lo) < len;
        f2 s = mul2(add2(om[pr], NX0), R);
        s.x = ok0 ? s.x : 0.0f;
        s.y = ok1 ? s.y : 0.0f;
        const f2 s2 = mul2(s, s), aa = mul2(s2, HS);
        const f2 t3 = mul2(aa, s), t4 = mul2(t3, s);
        const f2 ra4 = mul2(aa, R4);
        const f2 d3 = mul2(ra4, s), d2 = mul2(ra4, Q);
#pragma unroll
        for (int e = 0; e < 2; e++) {
            const int b = 2 * pr + e;
            const float c3 = e ? t3.y : t3.x, c4 = e ? t4.y : t4.x, g2 = e ? d2.y : d2.x, g3 = e ? d3.y : d3.x;
            a.T[b][0] = fma2(B01, dup(c3), a.T[b][0]); a.T[b][1] = fma2(B23, dup(c3), a.T[b][1]);
            a.D[b][0] = fma2(B01, dup(g2), a.D[b][0]); a.D[b][1] = fma2(B23, dup(g2), a.D[b][1]);
            a.T[b][0] = fma2(G01, dup(c4), a.T[b][0]); a.T[b][1] = fma2(G23, dup(c4), a.T[b][1]);
            a.D[b][0] = fma2(G01, dup(g3), a.D[b][0]); a.D[b][1] = fma2(G23, dup(g3), a.D[b][1]);
            if (HIGH) {   // Eq. 14c/e: the constant V_m inside [e3, e4)
                const float one = (e ? ok1 : ok0) ? 1.0f : 0.0f;
                a.T[b][0] = fma2(V01, dup(one), a.T[b][0]); a.T[b][1] = fma2(V23, dup(one), a.T[b][1]);
            }
        }
    }
}

// One mid entry: Eq. 13a-n for the lane's two energies E = om (packed), e2 <= E < e3 where ok; for an energy that
// is not ok all eight values are 0.  w[l] = w_l / V, dw[l] = (dw_l/dE) / V for the sorted corners; every quotient
// is a product of ratios bounded by 1 (G12); misprints read as in DESIGN.md (G3, G4).  Then the 4 x 8 projection.
__device__ __forceinline__ void eval_mid6(AccM6& acc, const float4 es, const float4 R, const uint32_t rng, const uint32_t pts,
                                          const f2 om, int bin0, const float4* __restrict__ sW4) {
    const int lo = (int)(rng & 0xffffu);
    const unsigned len = (rng >> 16) - (rng & 0xffffu);
    const bool oka = (unsigned)(bin0 - lo) < len, okb = (unsigned)(bin0 + 1 - lo) < len;
    const float e1 = es.x, e2 = es.y, e3 = es.z, e4 = es.w;
    const float i31 = R.x, i41 = R.y, i32 = R.z, i42 = R.w;
    const f2 NEG1 = dup(-1.0f), I41 = dup(i41), I31 = dup(i31), I32 = dup(i32), I42 = dup(i42);
    f2 Es, a;
    Es.x = oka ? om.x : e2;  Es.y = okb ? om.y : e2;
    a.x = oka ? Es.x - e1 : 0.0f;  a.y = okb ? Es.y - e1 : 0.0f;
    const f2 b = fma2(dup(e2), NEG1, Es);           // E - E2
    const f2 c = fma2(Es, NEG1, dup(e3));           // E3 - E
    const f2 d = fma2(Es, NEG1, dup(e4));           // E4 - E
    const f2 A31 = mul2(a, I31), A41 = mul2(a, I41);     // (E-E1)/E31, (E-E1)/E41
    const f2 B32 = mul2(b, I32), B42 = mul2(b, I42);     // (E-E2)/E32, (E-E2)/E42
    const f2 C31 = mul2(c, I31), C32 = mul2(c, I32);     // (E3-E)/E31, (E3-E)/E32
    const f2 D41 = mul2(d, I41), D42 = mul2(d, I42);     // (E4-E)/E41, (E4-E)/E42
    const f2 C1 = mul2(A31, A41);                                        // 13a
    const f2 dC1 = mul2(A31, dup(2.0f * i41));                           // 13b
    const f2 AB = mul2(A31, B32);
    const f2 C2 = mul2(mul2(A41, B32), C31);                             // 13c
    const f2 dC2 = mul2(I41, fma2(AB, NEG1, mul2(mul2(C32, add2(a, b)), I31)));   // 13d
    const f2 C3 = mul2(mul2(B32, B42), D41);                             // 13e
    const f2 dC3 = mul2(mul2(B32, I41), fma2(B42, NEG1, add2(D42, D42)));   // 13f
    const f2 C12 = add2(C1, C2), C23 = add2(C2, C3), C123 = add2(C12, C3);
    const f2 dC12 = add2(dC1, dC2), dC23 = add2(dC2, dC3), dC123 = add2(dC12, dC3);
    const f2 P = mul2(C12, C31), Q = mul2(C23, C32), Rr = mul2(C123, D41), Sx = mul2(C3, D42);
    const f2 dP = fma2(C12, dup(-i31), mul2(dC12, C31));   // d/dE [C12 (E3-E)/E31]
    const f2 dQ = fma2(C23, dup(-i32), mul2(dC23, C32));
    const f2 dR = fma2(C123, dup(-i41), mul2(dC123, D41));
    const f2 dS = fma2(C3, dup(-i42), mul2(dC3, D42));
    f2 w[4], dw[4];
    w[0] = add2(add2(C1, P), Rr);                            // 13g
    w[1] = add2(add2(C123, Q), Sx);                          // 13i
    w[2] = add2(fma2(P, NEG1, C12), fma2(Q, NEG1, C23));     // 13k (G3): (E-E1)/E31 = 1 - (E3-E)/E31
    w[3] = add2(fma2(Rr, NEG1, C123), fma2(Sx, NEG1, C3));   // 13m
    dw[0] = add2(add2(dC1, dP), dR);                         // 13h
    dw[1] = add2(add2(dC123, dQ), dS);                       // 13j
    dw[2] = add2(fma2(dP, NEG1, dC12), fma2(dQ, NEG1, dC23));   // 13l (G4)
    dw[3] = add2(fma2(dR, NEG1, dC123), fma2(dS, NEG1, dC3));   // 13n
#pragma unroll
    for (int l = 0; l < 4; l++) {   // Eq. 8 (:91): acc += b[l][:] * (dw[l], w[l])
        const unsigned pt = (pts >> (8 * l)) & 0xffu;
        const float4 v0 = sW4[2 * pt], v1 = sW4[2 * pt + 1];
        const f2 bb[4] = {make_float2(v0.x, v0.y), make_float2(v0.z, v0.w), make_float2(v1.x, v1.y), make_float2(v1.z, v1.w)};
#pragma unroll
        for (int j = 0; j < 4; j++) {
            acc.D[0][j] = fma2(bb[j], dup(dw[l].x), acc.D[0][j]);
            acc.D[1][j] = fma2(bb[j], dup(dw[l].y), acc.D[1][j]);
            acc.T[0][j] = fma2(bb[j], dup(w[l].x), acc.T[0][j]);
            acc.T[1][j] = fma2(bb[j], dup(w[l].y), acc.T[1][j]);
        }
    }
}

__device__ __forceinline__ int warp_incl_scan(int v, int lane) {
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int u = __shfl_up_sync(0xffffffffu, v, d);
        if (lane >= d) v += u;
    }
    return v;
}

// Warp 0 plans one pass over the chunks [0, NCH) that start at bin pb: truncates the pass to what the entry list
// holds, lays out the (kind, chunk) lists and deals the groups out to the chunks.
template <class C>
__device__ __forceinline__ void plan6(unsigned char* __restrict__ smem, int lane, int par) {
    constexpr int NCH = C::NCH;
    constexpr unsigned FULL = 0xffffffffu;
    int* sCnt = reinterpret_cast<int*>(smem + C::off_cnt) + par * 3 * NCH;
    int* sOff = reinterpret_cast<int*>(smem + C::off_off);
    int* sCur = reinterpret_cast<int*>(smem + C::off_cur);
    int* sGst = reinterpret_cast<int*>(smem + C::off_gst);
    int* sMisc = reinterpret_cast<int*>(smem + C::off_misc);
    int n[3][2];
#pragma unroll
    for (int k = 0; k < 3; k++) { n[k][0] = sCnt[k * NCH + lane]; n[k][1] = sCnt[k * NCH + 32 + lane]; }
    // chunks in order c = lane (first half), 32 + lane (second half); keep the longest prefix that fits the list
    const int t0 = n[0][0] + n[1][0] + n[2][0], t1 = n[0][1] + n[1][1] + n[2][1];
    const int inc0 = warp_incl_scan(t0, lane);
    const int inc1 = __shfl_sync(FULL, inc0, 31) + warp_incl_scan(t1, lane);
    const bool fit0 = inc0 <= C::CAP, fit1 = inc1 <= C::CAP;
    const int nc = __popc(__ballot_sync(FULL, fit0)) + __popc(__ballot_sync(FULL, fit1));   // >= 1: CAP >= 3 NTB
    if (!fit0) { n[0][0] = n[1][0] = n[2][0] = 0; }
    if (!fit1) { n[0][1] = n[1][1] = n[2][1] = 0; }
    // list layout: kind-major, chunk-minor
    int base = 0;
#pragma unroll
    for (int k = 0; k < 3; k++) {
        const int i0 = warp_incl_scan(n[k][0], lane);
        const int h0 = __shfl_sync(FULL, i0, 31);
        const int i1 = h0 + warp_incl_scan(n[k][1], lane);
        const int o0 = base + i0 - n[k][0], o1 = base + i1 - n[k][1];
        sOff[k * NCH + lane] = o0;  sCur[k * NCH + lane] = o0;
        sOff[k * NCH + 32 + lane] = o1;  sCur[k * NCH + 32 + lane] = o1;
        sCnt[k * NCH + lane] = n[k][0];  sCnt[k * NCH + 32 + lane] = n[k][1];
        base += __shfl_sync(FULL, i1, 31);
    }
    // groups per chunk: k_c = ceil(cost_c / lambda) with the smallest load lambda per group such that
    // sum_c k_c <= NG (bisection); the cost of an entry is ~ its instruction count (low 6 : high 7 : mid 16)
    const float c0 = (float)(6 * n[0][0] + 7 * n[1][0] + 16 * n[2][0]);
    const float c1 = (float)(6 * n[0][1] + 7 * n[1][1] + 16 * n[2][1]);
    float tot = c0 + c1;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) tot += __shfl_xor_sync(FULL, tot, d);
    const int nz = __popc(__ballot_sync(FULL, c0 > 0.0f)) + __popc(__ballot_sync(FULL, c1 > 0.0f));
    int k0 = 0, k1 = 0;
    if (nz > 0) {
        // lambda in [tot/NG, tot/(NG-nz)]: the upper end always fits (sum ceil(x) <= sum x + nz)
        float inv_hi = (float)C::NG / tot, inv_lo = (float)(C::NG - nz) / tot * 0.9999f;   // 1/lambda
#pragma unroll 1
        for (int it = 0; it < 9; ++it) {
            const bool last = (it == 8);
            const float inv = last ? inv_lo : 0.5f * (inv_lo + inv_hi);
            k0 = c0 > 0.0f ? max(1, (int)ceilf(c0 * inv)) : 0;
            k1 = c1 > 0.0f ? max(1, (int)ceilf(c1 * inv)) : 0;
            const int sum = __reduce_add_sync(FULL, k0 + k1);
            if (last) {
                if (sum > C::NG) { k0 = c0 > 0.0f ? 1 : 0; k1 = c1 > 0.0f ? 1 : 0; }   // cannot happen (rounding guard)
            } else if (sum <= C::NG) inv_lo = inv; else inv_hi = inv;
        }
    }
    const int g0 = warp_incl_scan(k0, lane);
    const int gh = __shfl_sync(FULL, g0, 31);
    const int g1 = gh + warp_incl_scan(k1, lane);
    sGst[lane] = g0 - k0;
    sGst[32 + lane] = g1 - k1;
    if (lane == 31) { sGst[NCH] = g1; sMisc[M6_NC] = nc; }
}

// count (FILL = false) or enter (FILL = true) the records of this thread into the (kind, chunk) lists of the pass
// [pb, pe); lin -> record STRIDE apart
template <class C, bool FILL>
__device__ __forceinline__ void scatter6(unsigned char* __restrict__ smem, int tid, int pb, int pe, int par) {
    const uint4* sRng = reinterpret_cast<const uint4*>(smem + C::off_rng);
    uint32_t* sEnt = reinterpret_cast<uint32_t*>(smem + C::off_ent);
    int* sCnt = reinterpret_cast<int*>(smem + C::off_cnt) + par * 3 * C::NCH;
    int* sCur = reinterpret_cast<int*>(smem + C::off_cur);
#pragma unroll 1
    for (int lin = tid; lin < C::NTB; lin += C::NT) {
        const uint32_t t = (uint32_t)(((unsigned)lin * (unsigned)C::STRIDE) % (unsigned)C::NTB);
        const uint4 rr4 = sRng[t];
#pragma unroll
        for (int k = 0; k < 3; k++) {
            const uint32_t rr = k == 0 ? rr4.x : k == 1 ? rr4.y : rr4.z;
            const int lo = (int)(rr & 0xffffu), hi = (int)(rr >> 16);
            if (lo < hi && hi > pb && lo < pe) {
                const uint32_t ent = t | ((k == 0 ? (rr4.w & 0xffu) : k == 1 ? (rr4.w >> 24) : 0u) << 16);
                const int cl = (min(hi, pe) - 1 - pb) >> 2;
                for (int c = (max(lo, pb) - pb) >> 2; c <= cl; ++c) {
                    if (FILL) sEnt[atomicAdd(&sCur[k * C::NCH + c], 1)] = ent;
                    else atomicAdd(&sCnt[k * C::NCH + c], 1);
                }
            }
        }
    }
}

// NORB = 8: the number of orbitals is fixed at compile time (all histogram offsets become immediates); 0: any
// multiple of 4.  BPS: blocks per SM the register budget is cut for.
template <int TX, int TY, int TZ, int NWARP, int NORB, int BPS>
__global__ void __launch_bounds__(NWARP * 32, BPS) tdos_main6(const MainParams p) {
    using C = Cfg6<TX, TY, TZ, NWARP>;
    constexpr int PX = C::PX, PY = C::PY, PK = C::PK, NTB = C::NTB, NT = C::NT, NCH = C::NCH, MB = C::MB;
    constexpr unsigned FULL = 0xffffffffu;

    extern __shared__ __align__(16) unsigned char smem[];
    float4* sLowS = reinterpret_cast<float4*>(smem + C::off_ls);
    float4* sLowG = reinterpret_cast<float4*>(smem + C::off_lg);
    float4* sHighS = reinterpret_cast<float4*>(smem + C::off_hs);
    float4* sHighG = reinterpret_cast<float4*>(smem + C::off_hg);
    float4* sHighV = reinterpret_cast<float4*>(smem + C::off_hv);
    float4* sMidE = reinterpret_cast<float4*>(smem + C::off_me);
    float4* sMidR = reinterpret_cast<float4*>(smem + C::off_mr);
    uint4* sRng = reinterpret_cast<uint4*>(smem + C::off_rng);
    const uint32_t* sEnt = reinterpret_cast<const uint32_t*>(smem + C::off_ent);
    int* sCntAll = reinterpret_cast<int*>(smem + C::off_cnt);
    const int* sOff = reinterpret_cast<const int*>(smem + C::off_off);
    const int* sGst = reinterpret_cast<const int*>(smem + C::off_gst);
    int* sMisc = reinterpret_cast<int*>(smem + C::off_misc);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, h = lane & 1;
    const int grp = warp * 16 + (lane >> 1);
    const int nE = p.nE, norb = NORB ? NORB : p.norb;
    const float* __restrict__ omega = p.omega;
    // the energy grid is probed 8 times per (tetrahedron, band): keep a block-wide copy in shared memory when it fits
    const float* om_loc = omega;
    if (p.om_smem) {
        float* sOmAll = reinterpret_cast<float*>(smem + C::bytes);
        for (int i = tid; i < nE; i += NT) sOmAll[i] = __ldg(omega + i);
        om_loc = sOmAll;
    }
    const float om0 = __ldg(omega);
    float inv_dom = 0.0f;
    if (nE > 1) {
        const float span = __ldg(omega + nE - 1) - om0;
        if (span > 0.0f) inv_dom = (float)(nE - 1) / span;
    }
    // rows [bin][ D | T | S ] of norb floats each, nEp = nE rounded up to 4 rows; blocks on one SM share a copy
    float* part = p.partial + (size_t)(blockIdx.x % p.nparts) * 3 * norb * p.nEp;
    const bool w_vec4 = !p.unitW && !p.cplx && p.sWm == 1 && ((reinterpret_cast<uintptr_t>(p.W) & 15) == 0) &&
                        (p.sWk % 4 == 0) && (p.sWn % 4 == 0);
    unsigned long long cnt_tb = 0, cnt_ev = 0, cnt_mid = 0;
#ifdef TDOS_PHASES
    long long ph_t[12] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0}, ph_last = clock64();
#define PH(k) do { const long long now_ = clock64(); ph_t[k] += now_ - ph_last; ph_last = now_; } while (0)
#else
#define PH(k) do { } while (0)
#endif

    // thread 0 draws the items and decodes them (orbital block, band fastest: neighbouring blocks share the tile's lines)
    auto next_item = [&](int* d) {
        const int item = (int)atomicAdd(p.next_item, 1u);
        d[M6_ITEM] = item;
        d[M6_LMAX] = -1;
        if (item < p.n_items) {
            int r = item;
            const int mb = r % p.nmb; r /= p.nmb;
            const int n = r % p.nb; r /= p.nb;
            const int tx = r % p.ntx; r /= p.ntx;
            const int ty = r % p.nty; r /= p.nty;
            d[M6_MB] = mb; d[M6_BAND] = n;
            d[M6_X0] = tx * TX; d[M6_Y0] = ty * TY; d[M6_Z0] = p.z_lo + r * TZ;
        }
    };
    // A1: stage the tile of the item described by d (periodic wrap: a tile never spans more than one period) into
    // buffer `buf`, asynchronously where the layout allows it (cp.async; complex input is squared on the way)
    auto stage = [&](const int* d, int buf) {
        const int x0 = d[M6_X0], y0 = d[M6_Y0], z0 = d[M6_Z0], n = d[M6_BAND], m0 = d[M6_MB] * MB;
        float* sE = reinterpret_cast<float*>(smem + C::off_e + buf * C::sz_e);
        float* sW = reinterpret_cast<float*>(smem + C::off_w + buf * C::sz_w);
        for (int qi = tid; qi < PK; qi += NT) {
            const int px = qi % PX, py = (qi / PX) % PY, pz = qi / (PX * PY);
            int gx = x0 + px, gy = y0 + py, gz = z0 + pz;
            while (gx >= p.N1) gx -= p.N1; while (gy >= p.N2) gy -= p.N2; while (gz >= p.N3) gz -= p.N3;
            const long long ik = gx + (long long)p.N1 * (gy + (long long)p.N2 * gz);
            cp_async4(sE + qi, p.E + ik * p.sEk + (long long)n * p.sEn);
        }
        if (p.unitW) {
            for (int qi = tid; qi < PK * MB; qi += NT) sW[qi] = ((qi % MB) + m0 < norb) ? 1.0f : 0.0f;
        } else if (w_vec4) {       // orbitals contiguous (AoS), whole float4s
            for (int qi = tid; qi < PK * 2; qi += NT) {
                const int part4 = qi & 1, k = qi >> 1;
                const int px = k % PX, py = (k / PX) % PY, pz = k / (PX * PY);
                int gx = x0 + px, gy = y0 + py, gz = z0 + pz;
                while (gx >= p.N1) gx -= p.N1; while (gy >= p.N2) gy -= p.N2; while (gz >= p.N3) gz -= p.N3;
                const long long ik = gx + (long long)p.N1 * (gy + (long long)p.N2 * gz);
                if (m0 + 4 * part4 < norb)
                    cp_async16(sW + k * MB + 4 * part4, p.W + ik * p.sWk + (long long)n * p.sWn + m0 + 4 * part4);
                else
                    *reinterpret_cast<float4*>(sW + k * MB + 4 * part4) = make_float4(0.f, 0.f, 0.f, 0.f);
            }
        } else {                   // any strides: AoS with unaligned rows, complex input, or SoA (k fastest across lanes)
            const bool kfast = p.sWm != 1;
            for (int qi = tid; qi < PK * MB; qi += NT) {
                const int k = kfast ? qi % PK : qi / MB, m = kfast ? qi / PK : qi % MB;
                const int px = k % PX, py = (k / PX) % PY, pz = k / (PX * PY);
                int gx = x0 + px, gy = y0 + py, gz = z0 + pz;
                while (gx >= p.N1) gx -= p.N1; while (gy >= p.N2) gy -= p.N2; while (gz >= p.N3) gz -= p.N3;
                const long long ik = gx + (long long)p.N1 * (gy + (long long)p.N2 * gz);
                const long long idx = ik * p.sWk + (long long)n * p.sWn + (long long)(m0 + m) * p.sWm;
                if (m0 + m >= norb) sW[k * MB + m] = 0.0f;
                else if (p.cplx) sW[k * MB + m] = load_weight(p, idx);
                else cp_async4(sW + k * MB + m, p.W + idx);
            }
        }
    };

    if (tid == 0) next_item(sMisc);
    for (int i = tid; i < 2 * 3 * NCH; i += NT) sCntAll[i] = 0;
    __syncthreads();
    if (sMisc[M6_ITEM] < p.n_items) stage(sMisc, 0);
    cp_async_wait_all();
    __syncthreads();
    for (int par = 0;; par ^= 1) {
        int* desc = sMisc + par * M6_DESC;          // this item
        int* dnext = sMisc + (par ^ 1) * M6_DESC;   // the next one
        if (desc[M6_ITEM] >= p.n_items) break;
        const int x0 = desc[M6_X0], y0 = desc[M6_Y0], z0 = desc[M6_Z0], mb = desc[M6_MB];
        const int m0 = mb * MB;
        const float* sE = reinterpret_cast<const float*>(smem + C::off_e + par * C::sz_e);
        const float4* sW4 = reinterpret_cast<const float4*>(smem + C::off_w + par * C::sz_w);
        int* sCnt = sCntAll + par * 3 * NCH;   // zero: cleared while the previous item was walked
        PH(0);
        if (tid == 0) next_item(dnext);        // read after barrier (2)

        // first bin of the item's span: no window starts below the first omega > (lowest energy of the tile)
        float emin = 3.0e38f;
        for (int qi = lane; qi < PK; qi += 32) emin = fminf(emin, sE[qi]);
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) emin = fminf(emin, __shfl_xor_sync(FULL, emin, d));
        int pb = locate6<true>(om_loc, nE, om0, inv_dom, emin) & ~(C::CH - 1);
        int pe = pb + C::NCHP * C::CH;
        PH(1);

        // ---- A2/A3 + record parameters: thread = (tetrahedron, band); counts of the first pass
        int lmax = -1;
#pragma unroll 1
        for (int t = tid; t < NTB; t += NT) {
            const int cube = t / 6, tet = t - cube * 6;
            const int cx = cube % TX, cy = (cube / TX) % TY, cz = cube / (TX * TY);
            const bool valid = (x0 + cx < p.N1) && (y0 + cy < p.N2) && (z0 + cz < p.z_hi);
            const int cbase = cx + PX * (cy + PY * cz);
            const int a0 = kTableI[tet][0], a1 = kTableI[tet][1], a2 = kTableI[tet][2], a3 = kTableI[tet][3];
            unsigned c0 = cbase + (a0 & 1) + PX * (((a0 >> 1) & 1) + PY * (a0 >> 2));
            unsigned c1 = cbase + (a1 & 1) + PX * (((a1 >> 1) & 1) + PY * (a1 >> 2));
            unsigned c2 = cbase + (a2 & 1) + PX * (((a2 >> 1) & 1) + PY * (a2 >> 2));
            unsigned c3 = cbase + (a3 & 1) + PX * (((a3 >> 1) & 1) + PY * (a3 >> 2));
            float e0 = sE[c0], e1 = sE[c1], e2 = sE[c2], e3 = sE[c3];
            TDOS_CSWAP(e0, e1, c0, c1);
            TDOS_CSWAP(e2, e3, c2, c3);
            TDOS_CSWAP(e0, e2, c0, c2);
            TDOS_CSWAP(e1, e3, c1, c3);
            TDOS_CSWAP(e1, e2, c1, c2);
            uint4 rr = make_uint4(0u, 0u, 0u, 0u);   // empty ranges
            if (valid) {
                // bins (reading G10): low [i1,i2), mid [i2,i3), high [i3,i4), full weight from i4 on
                const int i1 = locate6<true>(om_loc, nE, om0, inv_dom, e0);             // first omega > E1
                const int i2 = max(i1, locate6<false>(om_loc, nE, om0, inv_dom, e1));   // first omega >= E2
                const int i3 = max(i2, locate6<false>(om_loc, nE, om0, inv_dom, e2));
                const int i4 = max(i3, locate6<false>(om_loc, nE, om0, inv_dom, e3));
                rr = make_uint4((uint32_t)i1 | ((uint32_t)i2 << 16), (uint32_t)i3 | ((uint32_t)i4 << 16),
                                (uint32_t)i2 | ((uint32_t)i3 << 16), c0 | (c1 << 8) | (c2 << 16) | (c3 << 24));
                if (mb == 0) {   // work counters (exact integers; bench.py's flop count uses them)
                    cnt_tb += 1;
                    cnt_ev += (unsigned)(i4 - i1);
                    cnt_mid += (unsigned)(i3 - i2);
                }
                if (i1 < i4) lmax = max(lmax, i4 - 1);
                if (i1 < nE) {   // something of this tetrahedron is on the grid
                    // orbital weights of the sorted corners, packed along orbital pairs
                    f2 b[4][4];
#pragma unroll
                    for (int l = 0; l < 4; l++) {
                        const unsigned pt = l == 0 ? c0 : l == 1 ? c1 : l == 2 ? c2 : c3;
                        const float4 v0 = sW4[2 * pt], v1 = sW4[2 * pt + 1];
                        b[l][0] = make_float2(v0.x, v0.y); b[l][1] = make_float2(v0.z, v0.w);
                        b[l][2] = make_float2(v1.x, v1.y); b[l][3] = make_float2(v1.z, v1.w);
                    }
                    f2 V[4];
#pragma unroll
                    for (int j = 0; j < 4; j++) V[j] = add2(add2(b[0][j], b[1][j]), add2(b[2][j], b[3][j]));
                    // Eq. 15 (A6): from the first omega >= E4 on every corner carries the constant V:
                    // one add of sum_l b_l into the step histogram at bin i4 (prefix-summed in fp64 later)
                    if (i4 < nE) {
                        float* dst = part + (size_t)i4 * 3 * norb + 2 * norb + m0;
                        red_add4(dst, V[0].x, V[0].y, V[1].x, V[1].y);
                        if (m0 + 4 < norb) red_add4(dst + 4, V[2].x, V[2].y, V[3].x, V[3].y);
                    }
                    // reciprocals of the differences E_ij (Eq. 10); a vanishing difference is never USED by a
                    // non-empty interval (G11), clamping only keeps the unused values finite
                    const float tiny = 1e-30f;
                    const float e21 = e1 - e0, e43 = e3 - e2;
                    const float i21 = rcp_fast(fmaxf(e21, tiny)), i31 = rcp_fast(fmaxf(e2 - e0, tiny));
                    const float i41 = rcp_fast(fmaxf(e3 - e0, tiny)), i32 = rcp_fast(fmaxf(e2 - e1, tiny));
                    const float i42 = rcp_fast(fmaxf(e3 - e1, tiny)), i43 = rcp_fast(fmaxf(e43, tiny));
                    if (i1 < i2) {   // low record (Eq. 12): near corner 1, far corners 2, 3, 4 with ratios 1, qa, qb
                        const float qa = e21 * i31, qb = e21 * i41;
                        const f2 QA = dup(0.25f * qa), QB = dup(0.25f * qb), K = dup(-0.25f * (1.0f + qa + qb));
                        f2 G[4];
#pragma unroll
                        for (int j = 0; j < 4; j++)
                            G[j] = fma2(b[3][j], QB, fma2(b[2][j], QA, fma2(b[0][j], K, mul2(b[1][j], dup(0.25f)))));
                        sLowS[t] = make_float4(e0, i21, 4.0f * qa * qb, __uint_as_float(rr.x));
                        sLowG[2 * t] = make_float4(G[0].x, G[0].y, G[1].x, G[1].y);
                        sLowG[2 * t + 1] = make_float4(G[2].x, G[2].y, G[3].x, G[3].y);
                    }
                    if (i3 < i4) {   // high record (Eq. 14): near corner 4, far corners 3, 2, 1 with ratios 1, qa, qb
                        const float qa = e43 * i42, qb = e43 * i41;
                        const f2 QA = dup(0.25f * qa), QB = dup(0.25f * qb), K = dup(-0.25f * (1.0f + qa + qb));
                        f2 G[4];
#pragma unroll
                        for (int j = 0; j < 4; j++)
                            G[j] = fma2(b[0][j], QB, fma2(b[1][j], QA, fma2(b[3][j], K, mul2(b[2][j], dup(0.25f)))));
                        sHighS[t] = make_float4(e3, -i43, -4.0f * qa * qb, __uint_as_float(rr.y));
                        sHighG[2 * t] = make_float4(G[0].x, G[0].y, G[1].x, G[1].y);
                        sHighG[2 * t + 1] = make_float4(G[2].x, G[2].y, G[3].x, G[3].y);
                        sHighV[2 * t] = make_float4(V[0].x, V[0].y, V[1].x, V[1].y);
                        sHighV[2 * t + 1] = make_float4(V[2].x, V[2].y, V[3].x, V[3].y);
                    }
                    if (i2 < i3) {   // mid record (Eq. 13)
                        sMidE[t] = make_float4(e0, e1, e2, e3);
                        sMidR[t] = make_float4(i31, i41, i32, i42);
                    }
                    // entries of the first pass: the record of an interval overlaps the chunks of its bins
#pragma unroll
                    for (int k = 0; k < 3; k++) {
                        const int lo = k == 0 ? i1 : k == 1 ? i3 : i2, hi = k == 0 ? i2 : k == 1 ? i4 : i3;
                        if (lo < hi && lo < pe) {
                            const int cl = (min(hi, pe) - 1 - pb) >> 2;
                            for (int c = (lo - pb) >> 2; c <= cl; ++c) atomicAdd(&sCnt[k * NCH + c], 1);
                        }
                    }
                }
            }
            sRng[t] = rr;
        }
        lmax = __reduce_max_sync(FULL, lmax);
        if (lane == 0 && lmax >= 0) atomicMax(&desc[M6_LMAX], lmax);
        PH(2);
        __syncthreads();   // (2) records and first-pass counts complete; the next item's description is there
        const int bmax = desc[M6_LMAX];
        const bool more = dnext[M6_ITEM] < p.n_items;

        // ---- passes of up to NCHP chunks over the tile's energy span
        bool first = true;
        while (pb <= bmax) {
            if (!first) {
                for (int i = tid; i < 3 * NCH; i += NT) sCnt[i] = 0;
                __syncthreads();
                scatter6<C, false>(smem, tid, pb, pe, par);
                __syncthreads();
            }
            PH(3);
            if (warp == 0) plan6<C>(smem, lane, par);
            PH(4);
            if (first) {   // meanwhile: the next item's tile is on its way; its counters are cleared
                if (more) stage(dnext, par ^ 1);
                for (int i = tid; i < 3 * NCH; i += NT) sCntAll[(par ^ 1) * 3 * NCH + i] = 0;
            }
            first = false;
            PH(5);
            __syncthreads();   // (3)
            PH(6);
            const int pf = pb + sMisc[M6_NC] * C::CH;   // bins [pb, pf) are done in this pass
            scatter6<C, true>(smem, tid, pb, pf, par);
            PH(7);
            __syncthreads();   // (4)
            PH(8);

            // -- A4-A6: every group walks its share of its chunk's lists
            {
                // chunk of this group: the last c with sGst[c] <= grp
                int lo_c = 0, hi_c = NCH;   // invariant: sGst[lo_c] <= grp (sGst[0] = 0), answer in [lo_c, hi_c)
#pragma unroll
                for (int s = 0; s < 6; ++s) {
                    const int mid_c = (lo_c + hi_c) >> 1;
                    if (sGst[mid_c] <= grp) lo_c = mid_c; else hi_c = mid_c;
                }
                const int c = lo_c;
                const int gfirst = sGst[c], gk = sGst[c + 1] - gfirst;
                const bool has = grp < sGst[NCH] && gk > 0;
                const unsigned j = (unsigned)(grp - gfirst), kk = (unsigned)max(gk, 1);
                int ea[3], eb[3];
#pragma unroll
                for (int k = 0; k < 3; k++) {
                    const unsigned nn = has ? (unsigned)sCnt[k * NCH + c] : 0u;
                    const int o = sOff[k * NCH + c];
                    ea[k] = o + (int)((nn * j) / kk);
                    eb[k] = o + (int)((nn * (j + 1u)) / kk);
                }
                const int cb0 = pb + c * C::CH;   // first bin of the chunk
                f2 om4[2];
                om4[0] = make_float2(om_loc[min(cb0, nE - 1)], om_loc[min(cb0 + 1, nE - 1)]);
                om4[1] = make_float2(om_loc[min(cb0 + 2, nE - 1)], om_loc[min(cb0 + 3, nE - 1)]);
                // mid entries (Eq. 13): lane h takes the bins 2h, 2h+1 of the chunk, all 8 orbitals
                AccM6 accM;
                accM.zero();
                {
                    const int steps = __reduce_max_sync(FULL, eb[2] - ea[2]);
                    const f2 om = h ? om4[1] : om4[0];
                    int pp = ea[2];
                    uint32_t e = pp < eb[2] ? sEnt[pp] : 0u;
#pragma unroll 1
                    for (int s = 0; s < steps; ++s, ++pp) {
                        const uint32_t rec = e & 0xffffu;
                        const float4 es = sMidE[rec], R = sMidR[rec];
                        const uint4 rr = sRng[rec];
                        const bool act = pp < eb[2];
                        e = pp + 1 < eb[2] ? sEnt[pp + 1] : 0u;
                        if (act) eval_mid6(accM, es, R, rr.z, rr.w, om, cb0 + 2 * h, sW4);
                    }
                }
                // the low/high walk wants 4 bins x (orbitals 4h..4h+3) per lane: the partner's mid sums of this lane's
                // orbitals come over by shuffle
                AccE6 accE;
#pragma unroll
                for (int b = 0; b < 2; b++)
#pragma unroll
                    for (int jj = 0; jj < 2; jj++) {
                        // send: the pairs the partner owns (orbital pairs 2(1-h) + jj); keep: pairs 2h + jj
                        const f2 sd = h ? accM.D[b][jj] : accM.D[b][2 + jj], st = h ? accM.T[b][jj] : accM.T[b][2 + jj];
                        const f2 kd = h ? accM.D[b][2 + jj] : accM.D[b][jj], kt = h ? accM.T[b][2 + jj] : accM.T[b][jj];
                        f2 rd, rt;
                        rd.x = __shfl_xor_sync(FULL, sd.x, 1); rd.y = __shfl_xor_sync(FULL, sd.y, 1);
                        rt.x = __shfl_xor_sync(FULL, st.x, 1); rt.y = __shfl_xor_sync(FULL, st.y, 1);
                        // received: the partner's bins 2(1-h) + b; kept: this lane's bins 2h + b
                        accE.D[b][jj] = h ? rd : kd;      accE.T[b][jj] = h ? rt : kt;
                        accE.D[2 + b][jj] = h ? kd : rd;  accE.T[2 + b][jj] = h ? kt : rt;
                    }
                // low entries (Eq. 12); the parameters of the next entry are loaded while this one is evaluated
                {
                    const int steps = __reduce_max_sync(FULL, eb[0] - ea[0]);
                    int pp = ea[0];
                    uint32_t e = pp < eb[0] ? sEnt[pp] : 0u;
                    float4 S = sLowS[e & 0xffffu], G = sLowG[2 * (e & 0xffffu) + h], B = sW4[2 * (e >> 16) + h];
                    uint32_t e2 = pp + 1 < eb[0] ? sEnt[pp + 1] : 0u;
#pragma unroll 1
                    for (int s = 0; s < steps; ++s, ++pp) {
                        const float4 Sn = sLowS[e2 & 0xffffu], Gn = sLowG[2 * (e2 & 0xffffu) + h], Bn = sW4[2 * (e2 >> 16) + h];
                        e2 = pp + 2 < eb[0] ? sEnt[pp + 2] : 0u;
                        if (pp < eb[0]) eval_edge6<false>(accE, S, G, B, make_float4(0.f, 0.f, 0.f, 0.f), om4, cb0);
                        S = Sn; G = Gn; B = Bn;
                    }
                }
                // high entries (Eq. 14)
                {
                    const int steps = __reduce_max_sync(FULL, eb[1] - ea[1]);
                    int pp = ea[1];
                    uint32_t e = pp < eb[1] ? sEnt[pp] : 0u;
                    float4 S = sHighS[e & 0xffffu], G = sHighG[2 * (e & 0xffffu) + h], V = sHighV[2 * (e & 0xffffu) + h],
                           B = sW4[2 * (e >> 16) + h];
                    uint32_t e2 = pp + 1 < eb[1] ? sEnt[pp + 1] : 0u;
#pragma unroll 1
                    for (int s = 0; s < steps; ++s, ++pp) {
                        const float4 Sn = sHighS[e2 & 0xffffu], Gn = sHighG[2 * (e2 & 0xffffu) + h],
                                     Vn = sHighV[2 * (e2 & 0xffffu) + h], Bn = sW4[2 * (e2 >> 16) + h];
                        e2 = pp + 2 < eb[1] ? sEnt[pp + 2] : 0u;
                        if (pp < eb[1]) eval_edge6<true>(accE, S, G, B, V, om4, cb0);
                        S = Sn; G = Gn; B = Bn; V = Vn;
                    }
                }
                // flush: the chunk's rows (below nEp: the chunk holds a bin < nE), this lane's orbitals
                if (has && (eb[0] > ea[0] || eb[1] > ea[1] || eb[2] > ea[2]) && m0 + 4 * h < norb) {
#pragma unroll
                    for (int b = 0; b < 4; b++) {
                        float* row = part + (size_t)(cb0 + b) * 3 * norb + m0 + 4 * h;
                        red_add4(row, accE.D[b][0].x, accE.D[b][0].y, accE.D[b][1].x, accE.D[b][1].y);
                        red_add4(row + norb, accE.T[b][0].x, accE.T[b][0].y, accE.T[b][1].x, accE.T[b][1].y);
                    }
                }
            }
            pb = pf;
            pe = pb + C::NCHP * C::CH;
            PH(9);
            cp_async_wait_all();   // (the next item's tile has long arrived)
            PH(10);
            __syncthreads();       // (5) the next pass / item rewrites the lists and the records
        }
        if (first) {   // no window on the grid at all: the staging still has to happen
            if (more) stage(dnext, par ^ 1);
            for (int i = tid; i < 3 * NCH; i += NT) sCntAll[(par ^ 1) * 3 * NCH + i] = 0;
            cp_async_wait_all();
            __syncthreads();
        }
    }

#ifdef TDOS_PHASES
    if (lane == 0 && (warp == 0 || warp == NWARP - 1))
        for (int k = 0; k < 12; k++) atomicAdd(p.counters + 8 + (warp ? 12 : 0) + k, (unsigned long long)ph_t[k]);
#endif
    cnt_tb = __reduce_add_sync(FULL, (unsigned)cnt_tb);   // per warp < 2^32
    unsigned long long ev = cnt_ev, mid = cnt_mid;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        ev += __shfl_xor_sync(FULL, ev, d);
        mid += __shfl_xor_sync(FULL, mid, d);
    }
    if (lane == 0 && (cnt_tb | ev)) {
        atomicAdd(p.counters + 0, cnt_tb);
        atomicAdd(p.counters + 1, ev);
        atomicAdd(p.counters + 2, mid);
    }
}

}  // namespace tdos
