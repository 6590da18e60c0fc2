// tdos_kernels.cuh -- sm_100a kernels of the tetrahedron-DOS hot path.
//
// Main kernel `tdos_main`: persistent blocks; one work item = (tile of TX x TY x TZ cubes, band n,
// block of MB orbitals).  Per item:
//   A1/A2  the tile's (TX+1)(TY+1)(TZ+1) k-points of E (band n) and W (band n, MB orbitals) are
//          staged once in shared memory with periodic wrap -- tetrahedra are never materialised;
//          one thread per (tetrahedron, band) sorts its 4 corner energies (5 compare-exchanges
//          carrying the corner slots) and stores the record {e1..e4, 4 corner slots, bin window}.
//   A3     bin window: i1 = first bin with omega > e1, i4 = first bin with omega >= e4 -- exact,
//          decided on the fp32 omega values themselves.
//   A4-A6  every thread OWNS one energy bin of the tile's energy span and keeps its 2*MB sums
//          (DOS and in-window N) in registers: 8 consecutive lanes form a group that walks, on its
//          own, the records whose window overlaps the group's 8 bins; the record is a shared-memory
//          broadcast, the lane evaluates Eq. 12/13/14 at its own omega and does the 4 x MB
//          projection as FMAs into its registers.  No atomics, no write conflicts (the paper's
//          "thread = energy, thread-local accumulation", restricted to the window).
//          The Eq.-15 constant of finished tetrahedra goes into a block-local step histogram
//          (shared memory) at bin i4.
//   flush  registers + step histogram are added to this block's private partial histogram in HBM
//          (plain read-modify-write, the block is its only writer).
// `tdos_merge` sums the block partials in fp64; `tdos_finalize` prefix-sums the step histogram in
// fp64, scales by V and writes fp32 DOS and N (A7).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "tdos_weights.cuh"

namespace tdos {

struct MainParams {
    const float* E;
    const float* W;        // may be null when unitW
    const float* omega;
    long long sEk, sEn;          // E[ik*sEk + n*sEn]
    long long sWk, sWn, sWm;     // W[ik*sWk + n*sWn + m*sWm]
    int N1, N2, N3, nb, norb, nE;
    int z_lo, z_hi;              // cube slab [z_lo, z_hi)
    int ntx, nty, ntz;           // tiles per direction (z over the slab)
    int nmb;                     // orbital blocks of MB
    int n_items;                 // ntx*nty*ntz*nb*nmb
    int unitW;                   // W == 1
    float* partial;              // [gridDim.x][3][norb][nE]
    unsigned long long* counters;   // [0] n_tb, [1] n_eval = #(tb, omega) with E1 < omega < E4
};

// Table I of the paper, corner labels 1..8 -> 0..7; label c sits at offset
// (dx,dy,dz) = bits 0,1,2 of c (reading G7).
__device__ __constant__ int8_t kTableI[6][4] = {
    {0, 1, 2, 5}, {1, 2, 3, 5}, {0, 2, 4, 5}, {2, 3, 5, 7}, {2, 4, 5, 6}, {2, 5, 6, 7}};

// first index i in [0, nE] with omega[i] >= x (STRICT = false) or omega[i] > x (STRICT = true):
// direct index guess for a uniform grid, then an exact fix-up on the stored fp32 energies.
template <bool STRICT>
__device__ __forceinline__ int locate_bin(const float* __restrict__ omega, int nE, float om0, float inv_dom, float x) {
    float g = (x - om0) * inv_dom;
    g = fminf(fmaxf(g, 0.0f), (float)nE);
    int i = (int)g;
    if (STRICT) {
        while (i > 0 && __ldg(omega + i - 1) > x) --i;
        while (i < nE && __ldg(omega + i) <= x) ++i;
    } else {
        while (i > 0 && __ldg(omega + i - 1) >= x) --i;
        while (i < nE && __ldg(omega + i) < x) ++i;
    }
    return i;
}

#define TDOS_CSWAP(ea, eb, ca, cb)            \
    do {                                      \
        if (eb < ea) {                        \
            float te = ea; ea = eb; eb = te;  \
            unsigned tc = ca; ca = cb; cb = tc; \
        }                                     \
    } while (0)

template <int MB, int TX, int TY, int TZ>
struct TileCfg {
    static constexpr int PX = TX + 1, PY = TY + 1, PZ = TZ + 1;
    static constexpr int PK = PX * PY * PZ;          // k-points staged per tile
    static constexpr int NC = TX * TY * TZ;          // cubes per tile
    static constexpr int NTB = 6 * NC;               // (tetrahedron, band) records per item
    static_assert(NTB % 8 == 0, "records are scanned 8 at a time");
    static_assert(PK < 65536, "corner slots are 16-bit");
    // dynamic shared memory layout (byte offsets, 16-byte aligned pieces first)
    static constexpr size_t off_es = 0;                                   // float4 [NTB]
    static constexpr size_t off_w = off_es + sizeof(float4) * NTB;        // float  [PK*MB]
    static constexpr size_t off_cs = off_w + ((sizeof(float) * PK * MB + 15) / 16) * 16;   // uint2 [NTB]
    static constexpr size_t off_rng = off_cs + sizeof(uint2) * NTB;       // uint32 [NTB]
    static constexpr size_t off_e = off_rng + sizeof(uint32_t) * NTB;     // float  [PK]
    static constexpr size_t off_s = off_e + ((sizeof(float) * PK + 15) / 16) * 16;   // float [MB*NT], then int[2]
    static size_t bytes(int NT) { return off_s + sizeof(float) * MB * NT + 16; }
};

template <int MB, int TX, int TY, int TZ, int NT>
__global__ void __launch_bounds__(NT) tdos_main(const MainParams p) {
    using Cfg = TileCfg<MB, TX, TY, TZ>;
    constexpr int PX = Cfg::PX, PY = Cfg::PY, PK = Cfg::PK, NC = Cfg::NC, NTB = Cfg::NTB;
    extern __shared__ __align__(16) unsigned char smem[];
    float4* sEs = reinterpret_cast<float4*>(smem + Cfg::off_es);
    float* sW = reinterpret_cast<float*>(smem + Cfg::off_w);
    uint2* sCs = reinterpret_cast<uint2*>(smem + Cfg::off_cs);
    uint32_t* sRng = reinterpret_cast<uint32_t*>(smem + Cfg::off_rng);
    float* sE = reinterpret_cast<float*>(smem + Cfg::off_e);
    float* sS = reinterpret_cast<float*>(smem + Cfg::off_s);
    int* sMinMax = reinterpret_cast<int*>(sS + MB * NT);

    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int nE = p.nE;
    const float* __restrict__ omega = p.omega;
    const float om0 = __ldg(omega);
    float inv_dom = 0.0f;
    if (nE > 1) {
        const float span = __ldg(omega + nE - 1) - om0;
        if (span > 0.0f) inv_dom = (float)(nE - 1) / span;
    }
    float* part = p.partial + (size_t)blockIdx.x * 3 * p.norb * nE;   // written and re-read: no __restrict__
    const size_t qstride = (size_t)p.norb * nE;

    for (int item = blockIdx.x; item < p.n_items; item += gridDim.x) {
        // ---- decode the work item
        int r = item;
        const int mb = r % p.nmb; r /= p.nmb;
        const int n = r % p.nb; r /= p.nb;
        const int tx = r % p.ntx; r /= p.ntx;
        const int ty = r % p.nty; r /= p.nty;
        const int tz = r;
        const int x0 = tx * TX, y0 = ty * TY, z0 = p.z_lo + tz * TZ;
        const int m0 = mb * MB;

        if (tid == 0) { sMinMax[0] = 0x7fffffff; sMinMax[1] = -1; }

        // ---- A1/A2: stage the tile (periodic wrap), E then W
        for (int q = tid; q < PK; q += NT) {
            const int px = q % PX, py = (q / PX) % PY, pz = q / (PX * PY);
            const int gx = (x0 + px) % p.N1, gy = (y0 + py) % p.N2, gz = (z0 + pz) % p.N3;
            const long long ik = gx + (long long)p.N1 * (gy + (long long)p.N2 * gz);
            sE[q] = __ldg(p.E + ik * p.sEk + (long long)n * p.sEn);
        }
        if (p.unitW) {
            for (int q = tid; q < PK * MB; q += NT) sW[q] = ((q % MB) + m0 < p.norb) ? 1.0f : 0.0f;
        } else if (p.sWm == 1) {   // orbitals contiguous (AoS): m fastest across threads
            for (int q = tid; q < PK * MB; q += NT) {
                const int m = q % MB, k = q / MB;
                const int px = k % PX, py = (k / PX) % PY, pz = k / (PX * PY);
                const int gx = (x0 + px) % p.N1, gy = (y0 + py) % p.N2, gz = (z0 + pz) % p.N3;
                const long long ik = gx + (long long)p.N1 * (gy + (long long)p.N2 * gz);
                sW[k * MB + m] = (m0 + m < p.norb) ? __ldg(p.W + ik * p.sWk + (long long)n * p.sWn + (m0 + m)) : 0.0f;
            }
        } else {                   // k contiguous (SoA): k fastest across threads
            for (int q = tid; q < PK * MB; q += NT) {
                const int k = q % PK, m = q / PK;
                const int px = k % PX, py = (k / PX) % PY, pz = k / (PX * PY);
                const int gx = (x0 + px) % p.N1, gy = (y0 + py) % p.N2, gz = (z0 + pz) % p.N3;
                const long long ik = gx + (long long)p.N1 * (gy + (long long)p.N2 * gz);
                sW[k * MB + m] = (m0 + m < p.norb)
                                     ? __ldg(p.W + ik * p.sWk + (long long)n * p.sWn + (long long)(m0 + m) * p.sWm)
                                     : 0.0f;
            }
        }
        __syncthreads();

        // ---- A2/A3: one thread per (tetrahedron, band): sort, window, record
        {
            int lmin = 0x7fffffff, lmax = -1;
            unsigned cnt_tb = 0, cnt_ev = 0;
            for (int t = tid; t < NTB; t += NT) {
                const int tet = t / NC, cube = t - tet * NC;
                const int cx = cube % TX, cy = (cube / TX) % TY, cz = cube / (TX * TY);
                const bool valid = (x0 + cx < p.N1) && (y0 + cy < p.N2) && (z0 + cz < p.z_hi);
                const int cbase = cx + PX * (cy + PY * cz);
                unsigned c0, c1, c2, c3;
                {
                    const int a0 = kTableI[tet][0], a1 = kTableI[tet][1], a2 = kTableI[tet][2], a3 = kTableI[tet][3];
                    c0 = cbase + (a0 & 1) + PX * (((a0 >> 1) & 1) + PY * (a0 >> 2));
                    c1 = cbase + (a1 & 1) + PX * (((a1 >> 1) & 1) + PY * (a1 >> 2));
                    c2 = cbase + (a2 & 1) + PX * (((a2 >> 1) & 1) + PY * (a2 >> 2));
                    c3 = cbase + (a3 & 1) + PX * (((a3 >> 1) & 1) + PY * (a3 >> 2));
                }
                float e0 = sE[c0], e1 = sE[c1], e2 = sE[c2], e3 = sE[c3];
                TDOS_CSWAP(e0, e1, c0, c1);
                TDOS_CSWAP(e2, e3, c2, c3);
                TDOS_CSWAP(e0, e2, c0, c2);
                TDOS_CSWAP(e1, e3, c1, c3);
                TDOS_CSWAP(e1, e2, c1, c2);
                uint32_t rng = 0xffffffffu;
                if (valid) {
                    const int i1 = locate_bin<true>(omega, nE, om0, inv_dom, e0);      // first omega > E1
                    const int i4 = (e3 > e0) ? locate_bin<false>(omega, nE, om0, inv_dom, e3) : i1;   // first omega >= E4 (and > E1)
                    rng = (uint32_t)i1 | ((uint32_t)i4 << 16);
                    cnt_tb += 1;
                    cnt_ev += (unsigned)(i4 - i1);
                    if (i1 < nE) {
                        lmin = min(lmin, i1);
                        lmax = max(lmax, min(i4, nE - 1));
                    }
                }
                sEs[t] = make_float4(e0, e1, e2, e3);
                sCs[t] = make_uint2(c0 | (c1 << 16), c2 | (c3 << 16));
                sRng[t] = rng;
            }
            lmin = __reduce_min_sync(0xffffffffu, lmin);
            lmax = __reduce_max_sync(0xffffffffu, lmax);
            if (lane == 0 && lmax >= 0) {
                atomicMin(&sMinMax[0], lmin);
                atomicMax(&sMinMax[1], lmax);
            }
            if (mb == 0) {   // work counters (exact integers; bench.py's flop count uses them)
                cnt_tb = __reduce_add_sync(0xffffffffu, cnt_tb);
                cnt_ev = __reduce_add_sync(0xffffffffu, cnt_ev);
                if (lane == 0) {
                    atomicAdd(p.counters + 0, (unsigned long long)cnt_tb);
                    atomicAdd(p.counters + 1, (unsigned long long)cnt_ev);
                }
            }
        }
        __syncthreads();
        const int bmin = sMinMax[0], bmax = sMinMax[1];

        // ---- passes of NT bins over the tile's energy span
        for (int pb = bmin; pb <= bmax; pb += NT) {
            for (int q = tid; q < MB * NT; q += NT) sS[q] = 0.0f;
            __syncthreads();

            // Eq. 15 (A6): tetrahedra lying entirely below omega contribute V*sum_l b_l to every
            // higher bin: one add into the step histogram at bin i4
            for (int t = tid; t < NTB; t += NT) {
                const int i4 = (int)(sRng[t] >> 16);
                if (i4 < nE && i4 >= pb && i4 < pb + NT) {
                    const uint2 cs = sCs[t];
                    const float* b0 = sW + (cs.x & 0xffffu) * MB;
                    const float* b1 = sW + (cs.x >> 16) * MB;
                    const float* b2 = sW + (cs.y & 0xffffu) * MB;
                    const float* b3 = sW + (cs.y >> 16) * MB;
#pragma unroll
                    for (int m = 0; m < MB; m++) atomicAdd(&sS[m * NT + (i4 - pb)], (b0[m] + b1[m]) + (b2[m] + b3[m]));
                }
            }

            // A4-A6: thread = energy bin, group of 8 lanes = 8 consecutive bins
            const int bin = pb + tid;
            const float om = (bin < nE) ? __ldg(omega + bin) : -INFINITY;
            float accD[MB], accT[MB];
#pragma unroll
            for (int m = 0; m < MB; m++) accD[m] = accT[m] = 0.0f;

            const int gsh = lane & 24;
            const unsigned gmask = 0xffu << gsh;
            const int gl = lane & 7;
            const int gb = pb + (tid & ~7);
            if (gb <= bmax) {
                int t0 = 0, base = 0;
                unsigned mask = 0;
                for (;;) {
                    while (mask == 0 && t0 < NTB) {
                        const uint32_t rr = sRng[t0 + gl];
                        const int i1 = (int)(rr & 0xffffu), i4 = (int)(rr >> 16);
                        const bool hit = (i1 <= gb + 7) && (i4 > gb) && (i1 < i4);
                        mask = (__ballot_sync(gmask, hit) >> gsh) & 0xffu;
                        base = t0;
                        t0 += 8;
                    }
                    if (mask == 0) break;
                    const int t = base + __ffs(mask) - 1;
                    mask &= mask - 1;

                    const float4 es = sEs[t];
                    const uint2 cs = sCs[t];
                    float w[4], dw[4];
                    if (om > es.x && om < es.w) {
                        corner_weights_in_window(es.x, es.y, es.z, es.w, om, w, dw);
                    } else {
#pragma unroll
                        for (int l = 0; l < 4; l++) w[l] = dw[l] = 0.0f;
                    }
                    const unsigned cc[4] = {cs.x & 0xffffu, cs.x >> 16, cs.y & 0xffffu, cs.y >> 16};
#pragma unroll
                    for (int l = 0; l < 4; l++) {
                        const float* bp = sW + cc[l] * MB;
                        if constexpr (MB % 4 == 0) {
#pragma unroll
                            for (int m4 = 0; m4 < MB; m4 += 4) {
                                const float4 b = *reinterpret_cast<const float4*>(bp + m4);
                                accD[m4 + 0] = fmaf(b.x, dw[l], accD[m4 + 0]);
                                accD[m4 + 1] = fmaf(b.y, dw[l], accD[m4 + 1]);
                                accD[m4 + 2] = fmaf(b.z, dw[l], accD[m4 + 2]);
                                accD[m4 + 3] = fmaf(b.w, dw[l], accD[m4 + 3]);
                                accT[m4 + 0] = fmaf(b.x, w[l], accT[m4 + 0]);
                                accT[m4 + 1] = fmaf(b.y, w[l], accT[m4 + 1]);
                                accT[m4 + 2] = fmaf(b.z, w[l], accT[m4 + 2]);
                                accT[m4 + 3] = fmaf(b.w, w[l], accT[m4 + 3]);
                            }
                        } else {
#pragma unroll
                            for (int m = 0; m < MB; m++) {
                                const float b = bp[m];
                                accD[m] = fmaf(b, dw[l], accD[m]);
                                accT[m] = fmaf(b, w[l], accT[m]);
                            }
                        }
                    }
                }
            }
            __syncthreads();   // step histogram complete

            // ---- flush this pass into the block's private partial histogram
            if (bin <= bmax) {   // bmax <= nE-1
#pragma unroll
                for (int m = 0; m < MB; m++) {
                    if (m0 + m < p.norb) {
                        float* d = part + (size_t)(m0 + m) * nE + bin;
                        d[0] += accD[m];
                        d[qstride] += accT[m];
                        d[2 * qstride] += sS[m * NT + tid];
                    }
                }
            }
            __syncthreads();
        }
        __syncthreads();   // smem is reused by the next item
    }
}

// A7a: sum the block partials in fp64.  out[j] = sum_c partial[c][j], j < n (= 3*norb*nE)
__global__ void __launch_bounds__(256) tdos_merge(const float* __restrict__ partial, int nblk, size_t n, double* __restrict__ out) {
    for (size_t j = blockIdx.x * (size_t)blockDim.x + threadIdx.x; j < n; j += (size_t)gridDim.x * blockDim.x) {
        double s = 0.0;
        for (int c = 0; c < nblk; c++) s += (double)partial[(size_t)c * n + j];
        out[j] = s;
    }
}

// A7b: one block per orbital.  dos = V*D ; nos = V*(T + inclusive prefix over omega of S), fp64 inside.
__global__ void __launch_bounds__(1024) tdos_finalize(const double* __restrict__ part, int norb, int nE, double V,
                                                      float* __restrict__ dos, float* __restrict__ nos) {
    __shared__ double sh[1024];
    const int m = blockIdx.x, tid = threadIdx.x, nt = blockDim.x;
    const double* D = part + (size_t)m * nE;
    const double* T = part + ((size_t)norb + m) * nE;
    const double* S = part + ((size_t)2 * norb + m) * nE;
    const int chunk = (nE + nt - 1) / nt;
    const int lo = min(tid * chunk, nE), hi = min(lo + chunk, nE);
    double loc = 0.0;
    for (int i = lo; i < hi; i++) loc += S[i];
    sh[tid] = loc;
    __syncthreads();
    // inclusive Hillis-Steele scan over the per-thread chunk sums (fp64)
    for (int off = 1; off < nt; off <<= 1) {
        const double v = (tid >= off) ? sh[tid - off] : 0.0;
        __syncthreads();
        sh[tid] += v;
        __syncthreads();
    }
    double run = sh[tid] - loc;   // exclusive prefix of this chunk
    for (int i = lo; i < hi; i++) {
        run += S[i];
        dos[(size_t)m * nE + i] = (float)(V * D[i]);
        if (nos) nos[(size_t)m * nE + i] = (float)(V * (T[i] + run));
    }
}

// Register-resident FFMA chain: 8 independent accumulators per thread, ITER*8 FMAs (or FFMA2 pairs).
template <bool PACKED>
__global__ void __launch_bounds__(256) tdos_fma_probe(float* out, int iters, float a, float b) {
    float x[16];
#pragma unroll
    for (int i = 0; i < 16; i++) x[i] = (float)(threadIdx.x + i) * 1e-3f;
    if (PACKED) {
        unsigned long long av, bv, xv[8];
        asm("mov.b64 %0, {%1, %1};" : "=l"(av) : "f"(a));
        asm("mov.b64 %0, {%1, %1};" : "=l"(bv) : "f"(b));
#pragma unroll
        for (int i = 0; i < 8; i++) asm("mov.b64 %0, {%1, %2};" : "=l"(xv[i]) : "f"(x[2 * i]), "f"(x[2 * i + 1]));
        for (int it = 0; it < iters; it++) {
#pragma unroll
            for (int i = 0; i < 8; i++) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(xv[i]) : "l"(av), "l"(bv));
        }
#pragma unroll
        for (int i = 0; i < 8; i++) asm("mov.b64 {%0, %1}, %2;" : "=f"(x[2 * i]), "=f"(x[2 * i + 1]) : "l"(xv[i]));
    } else {
        for (int it = 0; it < iters; it++) {
#pragma unroll
            for (int i = 0; i < 16; i++) x[i] = fmaf(x[i], a, b);
        }
    }
    float s = 0.0f;
#pragma unroll
    for (int i = 0; i < 16; i++) s += x[i];
    if (s == 12345.678f) out[0] = s;   // keep the chain alive
}

}  // namespace tdos
