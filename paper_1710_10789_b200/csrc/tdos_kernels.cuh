// tdos_kernels.cuh -- sm_100a kernels of the tetrahedron-DOS hot path.
//
// Main kernel `tdos_main`: one persistent block per SM; every WARP is an autonomous worker with its
// own slice of shared memory (no block barriers at all).  One work item = (tile of TX x TY x TZ cubes,
// band n, block of MB orbitals).  Per item, a warp does
//   A1/A2  stage the tile's (TX+1)(TY+1)(TZ+1) k-points of E (band n) and W (band n, MB orbitals) in
//          its shared-memory slice, with periodic wrap -- tetrahedra are never materialised; lane =
//          (tetrahedron, band) record: sort the 4 corner energies (5 compare-exchanges carrying the
//          corner slots), store {e1..e4, 4 corner slots};
//   A3     bin window: i1 = first bin with omega > e1, i4 = first bin with omega >= e4 -- exact,
//          decided on the fp32 omega values themselves;
//   A6'    Eq. 15: the constant sum_l b_l of a finished tetrahedron goes, as ONE vector reduction per
//          record, into the block's step histogram S[i4][m] (prefix-summed later in fp64);
//   A4-A6  the paper's "thread = energy, thread-local accumulation" restricted to the
//          window: lanes OWN energy bins and keep 2*MB sums (DOS and in-window N) in registers.  A warp
//          is NG groups of GL lanes; a group owns GL consecutive bins (a "chunk") at a time.  Which
//          records overlap which chunk is a bitmap built with warp ballots; the (record, chunk) entries
//          of the whole item are split EVENLY over the NG groups (prefix sum over chunks), so the groups
//          of a warp run the same number of steps.  Per step a group fetches its next record (a
//          shared-memory broadcast), every lane evaluates Eq. 12/13/14 at its own omega and does the
//          4 x MB projection as FMAs into its registers.  When a group leaves a chunk it adds its
//          registers to the block's partial histogram (fp32 reductions in L2, one coalesced sector
//          per orbital).
// `tdos_merge` sums the block partials in fp64; `tdos_finalize` prefix-sums the step histogram in
// fp64, scales by V and writes fp32 DOS and N (A7).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>

#include "tdos_weights.cuh"

namespace tdos {

struct MainParams {
    const float* E;
    const float* W;        // may be null when unitW
    const float* omega;
    long long sEk, sEn;          // E[ik*sEk + n*sEn]
    long long sWk, sWn, sWm;     // W[ik*sWk + n*sWn + m*sWm]
    int N1, N2, N3, nb, norb, nE;
    int nEp;                     // rows per block in `partial` (nE, or nE rounded up to 4 for tdos_main5)
    int z_lo, z_hi;              // cube slab [z_lo, z_hi)
    int ntx, nty, ntz;           // tiles per direction (z over the slab)
    int nmb;                     // orbital blocks of MB
    int n_items;                 // ntx*nty*ntz*nb*nmb
    int unitW;                   // W == 1
    // orbital selection (tetra_dos_select; "five Fe 3d orbitals ... and the total"): nsel > 0 or
    // total: output row j < nsel is input orbital sel[j], row nsel (if total) is the sum over all norb_in input
    // orbitals, the rows up to norb are zero padding.  Otherwise output row = input orbital.
    int nsel, total, norb_in;
    short sel[32];
    int cplx;                    // W holds complex eigenvector elements a (re, im pairs), strides count pairs: b = |a|^2
    int om_smem;                 // tdos_main5: the launch has room for a copy of omega behind the warps' slices
    int w64;                     // tdos_main<..., ACC64 = true> only: corner weights in double precision too
    // kernel choice on the device (null: this kernel runs): {sum of window lengths in bins, (tetrahedron, band) pairs}
    // of a sample, written by tdos_estimate earlier on the stream; see wanted_generation()
    const unsigned long long* est;
    float* partial;              // [gridDim.x] rows [nEp][ D(norb) | T(norb) | S(norb) ]
    double* partial64;           // the same in fp64 (tdos_main<..., ACC64 = true>: "switch to double precision")
    unsigned int* next_item;        // tdos_main5: work counter, zero at launch
    unsigned long long* counters;   // [0] n_tb, [1] n_eval = #(tb, omega) with E1 < omega < E4
};

// Mean number of bins with E1 < omega < E4 per (tetrahedron, band) below which tdos_main (generation 3: one record per
// tetrahedron, groups of one lane = chunks of 2 bins) beats tdos_main5 (generation 5: one record per interval of
// Eq. 12-14, chunks of 4 bins) -- config 5's windows are 3 bins.  Measured on the Nk = 64 grid: 6.6 bins 1.20 against
// 1.24 ms, 8.4 bins 1.42 against 1.37 ms.
constexpr unsigned long long kShortWindowBins = 7;
__host__ __device__ __forceinline__ int wanted_generation(unsigned long long sum_bins, unsigned long long n_tb) {
    return (n_tb > 0 && sum_bins < kShortWindowBins * n_tb) ? 3 : 5;
}

// Table I of the paper, corner labels 1..8 -> 0..7; label c sits at offset
// (dx,dy,dz) = bits 0,1,2 of c (reading G7).
__device__ __constant__ int8_t kTableI[6][4] = {
    {0, 1, 2, 5}, {1, 2, 3, 5}, {0, 2, 4, 5}, {2, 3, 5, 7}, {2, 4, 5, 6}, {2, 5, 6, 7}};

// b_{n,m}(k) = |a_n^m(k)|^2 (Eq. 3, :48; the paper ships re and im separately, :263) or the weight itself
__device__ __forceinline__ float load_weight(const MainParams& p, long long idx) {
    if (p.cplx) {
        const float2 a = __ldg(reinterpret_cast<const float2*>(p.W) + idx);
        return fmaf(a.x, a.x, a.y * a.y);
    }
    return __ldg(p.W + idx);
}

// weight of OUTPUT row j (< p.norb) at the k-point/band whose orbital 0 sits at `base`
__device__ __forceinline__ float load_out_weight(const MainParams& p, long long base, int j) {
    if (p.nsel == 0 && !p.total) return load_weight(p, base + (long long)j * p.sWm);
    if (j < p.nsel) return load_weight(p, base + (long long)p.sel[j] * p.sWm);
    float s = 0.0f;
    if (j == p.nsel && p.total)
        for (int m = 0; m < p.norb_in; m++) s += load_weight(p, base + (long long)m * p.sWm);
    return s;
}

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

// i1 = first omega > e_lo, i4 = first omega >= e_hi (or i1 if the two energies coincide) on an energy array in any
// address space: both index guesses and the four energies next to them are fetched before any is looked at, so the
// loads overlap; the exact fix-up loops only run where a guess is off by more than its own bin.
__device__ __forceinline__ void locate_window(const float* om, int nE, float om0, float inv_dom, float e_lo, float e_hi,
                                              int& i1, int& i4) {
    float g1 = fminf(fmaxf((e_lo - om0) * inv_dom, 0.0f), (float)nE), g4 = fminf(fmaxf((e_hi - om0) * inv_dom, 0.0f), (float)nE);
    int a = (int)g1, b = (int)g4;
    const float a0 = om[max(a - 1, 0)], a1 = om[min(a, nE - 1)], b0 = om[max(b - 1, 0)], b1 = om[min(b, nE - 1)];
    if (a > 0 && a0 > e_lo) { --a; while (a > 0 && om[a - 1] > e_lo) --a; }
    else if (a < nE && a1 <= e_lo) { ++a; while (a < nE && om[a] <= e_lo) ++a; }
    if (b > 0 && b0 >= e_hi) { --b; while (b > 0 && om[b - 1] >= e_hi) --b; }
    else if (b < nE && b1 < e_hi) { ++b; while (b < nE && om[b] < e_hi) ++b; }
    i1 = a;
    i4 = (e_hi > e_lo) ? b : a;
}

#define TDOS_CSWAP(ea, eb, ca, cb)            \
    do {                                      \
        if (eb < ea) {                        \
            float te = ea; ea = eb; eb = te;  \
            unsigned tc = ca; ca = cb; cb = tc; \
        }                                     \
    } while (0)

// fire-and-forget fp32 reductions into global memory (performed in L2)
__device__ __forceinline__ void red_add(float* addr, float v) {
    asm volatile("red.global.add.f32 [%0], %1;" ::"l"(addr), "f"(v) : "memory");
}
__device__ __forceinline__ void red_add4(float* addr, float a, float b, float c, float d) {   // 16-byte aligned
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}

__device__ __forceinline__ void red_add2(float* addr, float a, float b) {   // 8-byte aligned
    asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(addr), "f"(a), "f"(b) : "memory");
}

// Per-warp shared-memory slice.
template <int MB, int TX, int TY, int TZ>
struct WarpCfg {
    static constexpr int PX = TX + 1, PY = TY + 1, PZ = TZ + 1;
    static constexpr int PK = PX * PY * PZ;          // k-points staged per tile
    static constexpr int NC = TX * TY * TZ;          // cubes per tile
    static constexpr int NTB = 6 * NC;               // (tetrahedron, band) records per item
    static constexpr int NWORD = (NTB + 31) / 32;    // 32-record words of a chunk's bitmap
    static constexpr int BST = NWORD | 1;            // odd word stride between chunks: conflict-free column stores
    static constexpr int NCH = 32;                   // chunks per pass (lane c keeps chunk c's counters)
    static constexpr int WST = (MB >= 4) ? MB + 4 : MB;   // floats between k-points in sW: 48-byte rows spread the banks
    static_assert(NWORD <= 32, "word mask is 32 bits");
    static_assert(PK * WST < 65536, "corner slots are 16-bit");
    static constexpr size_t a16(size_t x) { return (x + 15) / 16 * 16; }
    static constexpr size_t off_es = 0;                                        // float4 [NWORD*32]
    static constexpr size_t off_w = off_es + sizeof(float4) * NWORD * 32;      // float  [PK*WST]
    static constexpr size_t off_cs = off_w + a16(sizeof(float) * PK * WST);    // uint2  [NWORD*32]
    static constexpr size_t off_rng = off_cs + sizeof(uint2) * NWORD * 32;     // uint32 [NWORD*32]
    static constexpr size_t off_e = off_rng + sizeof(uint32_t) * NWORD * 32;   // float  [PK]
    static constexpr size_t off_bm = off_e + a16(sizeof(float) * PK);          // uint32 [NCH*BST]
    static constexpr size_t off_off = off_bm + a16(sizeof(uint32_t) * NCH * BST);   // int [NCH], uint32 wordmask [NCH]
    static constexpr size_t bytes = off_off + a16(sizeof(int) * 2 * NCH);
};

template <int MB>
__device__ __forceinline__ void load_b(const float* __restrict__ bp, float (&b)[MB]) {
    if constexpr (MB % 4 == 0) {
#pragma unroll
        for (int m4 = 0; m4 < MB; m4 += 4) {
            const float4 v = *reinterpret_cast<const float4*>(bp + m4);
            b[m4] = v.x; b[m4 + 1] = v.y; b[m4 + 2] = v.z; b[m4 + 3] = v.w;
        }
    } else if constexpr (MB == 2) {
        const float2 v = *reinterpret_cast<const float2*>(bp);
        b[0] = v.x; b[1] = v.y;
    } else {
#pragma unroll
        for (int m = 0; m < MB; m++) b[m] = bp[m];
    }
}

// Register accumulators of one lane: two adjacent energy bins (a, b) x MB orbitals x {DOS, in-window N}.
// MB >= 2: packed along the orbitals, acc[bin][m/2] = (m, m+1);  MB == 1: packed along the bins.
template <int MB>
struct Acc {
    static constexpr int NP = (MB >= 2) ? MB / 2 : 1;
    f2 D[2][NP], T[2][NP];
    __device__ __forceinline__ void zero() {
#pragma unroll
        for (int h = 0; h < 2; h++)
#pragma unroll
            for (int j = 0; j < NP; j++) D[h][j] = T[h][j] = make_float2(0.f, 0.f);
    }
    // acc += b[l][:] * (dw[l], w[l]) for the 4 sorted corners; w, dw packed along the two bins
    __device__ __forceinline__ void project(const float* __restrict__ sW, const unsigned (&cc)[4], const f2 (&w)[4],
                                            const f2 (&dw)[4]) {
#pragma unroll
        for (int l = 0; l < 4; l++) {
            float b[MB];
            load_b<MB>(sW + cc[l], b);
            if constexpr (MB >= 2) {
                const f2 da = dup(dw[l].x), db = dup(dw[l].y), wa = dup(w[l].x), wb = dup(w[l].y);
#pragma unroll
                for (int j = 0; j < NP; j++) {
                    const f2 bb = make_float2(b[2 * j], b[2 * j + 1]);
                    D[0][j] = fma2(bb, da, D[0][j]);
                    D[1][j] = fma2(bb, db, D[1][j]);
                    T[0][j] = fma2(bb, wa, T[0][j]);
                    T[1][j] = fma2(bb, wb, T[1][j]);
                }
            } else {
                const f2 bb = dup(b[0]);
                D[0][0] = fma2(bb, dw[l], D[0][0]);
                T[0][0] = fma2(bb, w[l], T[0][0]);
            }
        }
    }
    // add to the block's partial histogram rows [bin][ D(norb) | T(norb) | S(norb) ] and clear
    __device__ __forceinline__ void flush(float* __restrict__ part, int bin0, int nE, int norb, int m0, bool vec4) {
        if constexpr (MB >= 2) {
#pragma unroll
            for (int h = 0; h < 2; h++) {
                if (bin0 + h < nE) {
                    float* row = part + (size_t)(bin0 + h) * 3 * norb + m0;
                    if (vec4) {
                        if constexpr (MB % 4 == 0) {
#pragma unroll
                            for (int j = 0; j < NP; j += 2) {
                                if (m0 + 2 * j < norb) {
                                    red_add4(row + 2 * j, D[h][j].x, D[h][j].y, D[h][j + 1].x, D[h][j + 1].y);
                                    red_add4(row + norb + 2 * j, T[h][j].x, T[h][j].y, T[h][j + 1].x, T[h][j + 1].y);
                                }
                            }
                        }
                    } else {
#pragma unroll
                        for (int j = 0; j < NP; j++) {
                            if (m0 + 2 * j < norb) { red_add(row + 2 * j, D[h][j].x); red_add(row + norb + 2 * j, T[h][j].x); }
                            if (m0 + 2 * j + 1 < norb) { red_add(row + 2 * j + 1, D[h][j].y); red_add(row + norb + 2 * j + 1, T[h][j].y); }
                        }
                    }
                }
            }
        } else {
            if (bin0 < nE) {
                float* row = part + (size_t)bin0 * 3 * norb + m0;
                red_add(row, D[0][0].x);
                red_add(row + norb, T[0][0].x);
            }
            if (bin0 + 1 < nE) {
                float* row = part + (size_t)(bin0 + 1) * 3 * norb + m0;
                red_add(row, D[0][0].y);
                red_add(row + norb, T[0][0].y);
            }
        }
        zero();
    }
};

// fp64 accumulation ("one can in principle switch to double precision"): the corner weights stay the
// paper's single-precision arithmetic, every SUM taken after them -- registers, block partials, step histogram,
// merge -- is fp64.  Same interface as Acc<MB>.
__device__ __forceinline__ void red_add_f64(double* addr, double v) {
    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(addr), "d"(v) : "memory");
}
template <int MB>
struct Acc64 {
    double D[2][MB], T[2][MB];
    __device__ __forceinline__ void zero() {
#pragma unroll
        for (int h = 0; h < 2; h++)
#pragma unroll
            for (int m = 0; m < MB; m++) D[h][m] = T[h][m] = 0.0;
    }
    __device__ __forceinline__ void project(const float* __restrict__ sW, const unsigned (&cc)[4], const f2 (&w)[4],
                                            const f2 (&dw)[4]) {
#pragma unroll
        for (int l = 0; l < 4; l++) {
            float b[MB];
            load_b<MB>(sW + cc[l], b);
            const double da = (double)dw[l].x, db = (double)dw[l].y, wa = (double)w[l].x, wb = (double)w[l].y;
#pragma unroll
            for (int m = 0; m < MB; m++) {
                const double bm = (double)b[m];
                D[0][m] = fma(bm, da, D[0][m]);
                D[1][m] = fma(bm, db, D[1][m]);
                T[0][m] = fma(bm, wa, T[0][m]);
                T[1][m] = fma(bm, wb, T[1][m]);
            }
        }
    }
    // the same with double-precision weights, [l][energy]
    __device__ __forceinline__ void project64(const float* __restrict__ sW, const unsigned (&cc)[4], const double (&w)[4][2],
                                              const double (&dw)[4][2]) {
#pragma unroll
        for (int l = 0; l < 4; l++) {
            float b[MB];
            load_b<MB>(sW + cc[l], b);
#pragma unroll
            for (int m = 0; m < MB; m++) {
                const double bm = (double)b[m];
                D[0][m] = fma(bm, dw[l][0], D[0][m]);
                D[1][m] = fma(bm, dw[l][1], D[1][m]);
                T[0][m] = fma(bm, w[l][0], T[0][m]);
                T[1][m] = fma(bm, w[l][1], T[1][m]);
            }
        }
    }
    __device__ __forceinline__ void flush(double* __restrict__ part, int bin0, int nE, int norb, int m0, bool) {
#pragma unroll
        for (int h = 0; h < 2; h++) {
            if (bin0 + h < nE) {
                double* row = part + (size_t)(bin0 + h) * 3 * norb + m0;
#pragma unroll
                for (int m = 0; m < MB; m++)
                    if (m0 + m < norb) { red_add_f64(row + m, D[h][m]); red_add_f64(row + norb + m, T[h][m]); }
            }
        }
        zero();
    }
};

template <int MB, int TX, int TY, int TZ, int GL, int NWARP, bool ACC64 = false>
__global__ void __launch_bounds__(NWARP * 32, 1) tdos_main(const MainParams p) {
    using Cfg = WarpCfg<MB, TX, TY, TZ>;
    constexpr int PX = Cfg::PX, PY = Cfg::PY, PK = Cfg::PK, NC = Cfg::NC, NTB = Cfg::NTB;
    constexpr int NWORD = Cfg::NWORD, BST = Cfg::BST, NCH = Cfg::NCH, WST = Cfg::WST;
    constexpr int NG = 32 / GL;             // groups per warp
    constexpr int CH = 2 * GL;              // bins per chunk: every lane owns two adjacent bins
    constexpr int PASS = NCH * CH;          // bins per pass
    constexpr unsigned FULL = 0xffffffffu;
    static_assert(GL == 1 || GL == 2 || GL == 4 || GL == 8 || GL == 16, "group width");

    extern __shared__ __align__(16) unsigned char smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned char* base = smem + (size_t)warp * Cfg::bytes;
    float4* sEs = reinterpret_cast<float4*>(base + Cfg::off_es);
    float* sW = reinterpret_cast<float*>(base + Cfg::off_w);
    uint2* sCs = reinterpret_cast<uint2*>(base + Cfg::off_cs);
    uint32_t* sRng = reinterpret_cast<uint32_t*>(base + Cfg::off_rng);
    float* sE = reinterpret_cast<float*>(base + Cfg::off_e);
    uint32_t* sBm = reinterpret_cast<uint32_t*>(base + Cfg::off_bm);
    int* sOff = reinterpret_cast<int*>(base + Cfg::off_off);
    uint32_t* sWm = reinterpret_cast<uint32_t*>(sOff + NCH);

    if (p.est && wanted_generation(p.est[0], p.est[1]) != 3) return;   // the other kernel of the pair runs
    const int nE = p.nE;
    const int norb = p.norb;
    const float* __restrict__ omega = p.omega;
    // the energy grid is probed 4 times per (tetrahedron, band): keep a block-wide copy in shared memory when it fits
    const float* om_loc = omega;
    if (p.om_smem) {
        float* sOmAll = reinterpret_cast<float*>(smem + (size_t)NWARP * Cfg::bytes);
        for (int i = threadIdx.x; i < nE; i += NWARP * 32) sOmAll[i] = __ldg(omega + i);
        __syncthreads();
        om_loc = sOmAll;
    }
    const float om0 = __ldg(omega);
    float inv_dom = 0.0f;
    if (nE > 1) {
        const float span = __ldg(omega + nE - 1) - om0;
        if (span > 0.0f) inv_dom = (float)(nE - 1) / span;
    }
    // rows [bin][ D | T | S ] of this block's partial histogram, fp32 or (ACC64) fp64
    using part_t = typename std::conditional<ACC64, double, float>::type;
    part_t* part;
    if constexpr (ACC64) part = p.partial64 + (size_t)blockIdx.x * 3 * norb * p.nEp;
    else part = p.partial + (size_t)blockIdx.x * 3 * norb * p.nEp;
    const bool vec4 = (MB % 4 == 0) && (norb % 4 == 0);          // 16-byte aligned vector reductions
    const bool w_vec4 = (MB % 4 == 0) && !p.unitW && !p.cplx && p.sWm == 1 && (norb % 4 == 0) && p.nsel == 0 && !p.total &&
                        ((reinterpret_cast<uintptr_t>(p.W) & 15) == 0);

    const int g = lane / GL, gl = lane % GL;
    unsigned long long cnt_tb = 0, cnt_ev = 0;
    const float qnan = __int_as_float(0x7fc00000);

    const int gwarp = blockIdx.x * NWARP + warp, nwarps = gridDim.x * NWARP;
    for (int item = gwarp; item < p.n_items; item += nwarps) {
        // ---- decode the work item (orbital block, band fastest: neighbouring warps share the tile's lines)
        int r = item;
        const int mb = r % p.nmb; r /= p.nmb;
        const int n = r % p.nb; r /= p.nb;
        const int tx = r % p.ntx; r /= p.ntx;
        const int ty = r % p.nty; r /= p.nty;
        const int tz = r;
        const int x0 = tx * TX, y0 = ty * TY, z0 = p.z_lo + tz * TZ;
        const int m0 = mb * MB;

        // ---- A1/A2: stage the tile (periodic wrap), E then W
        for (int q = lane; q < PK; q += 32) {
            const int px = q % PX, py = (q / PX) % PY, pz = q / (PX * PY);
            const int gx = (x0 + px) % p.N1, gy = (y0 + py) % p.N2, gz = (z0 + pz) % p.N3;
            const long long ik = gx + (long long)p.N1 * (gy + (long long)p.N2 * gz);
            sE[q] = __ldg(p.E + ik * p.sEk + (long long)n * p.sEn);
        }
        if (p.unitW) {
            for (int q = lane; q < PK * MB; q += 32) sW[(q / MB) * WST + q % MB] = ((q % MB) + m0 < norb) ? 1.0f : 0.0f;
        } else if (w_vec4) {       // orbitals contiguous (AoS), whole float4s
            constexpr int Q4 = (MB >= 4) ? MB / 4 : 1;
            for (int q = lane; q < PK * Q4; q += 32) {
                const int part4 = q % Q4, k = q / Q4;
                const int px = k % PX, py = (k / PX) % PY, pz = k / (PX * PY);
                const int gx = (x0 + px) % p.N1, gy = (y0 + py) % p.N2, gz = (z0 + pz) % p.N3;
                const long long ik = gx + (long long)p.N1 * (gy + (long long)p.N2 * gz);
                float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
                if (m0 + 4 * part4 < norb)
                    v = __ldg(reinterpret_cast<const float4*>(p.W + ik * p.sWk + (long long)n * p.sWn + m0 + 4 * part4));
                *reinterpret_cast<float4*>(sW + k * WST + 4 * part4) = v;
            }
        } else if (p.sWm == 1) {   // orbitals contiguous (AoS): m fastest across lanes
            for (int q = lane; q < PK * MB; q += 32) {
                const int m = q % MB, k = q / MB;
                const int px = k % PX, py = (k / PX) % PY, pz = k / (PX * PY);
                const int gx = (x0 + px) % p.N1, gy = (y0 + py) % p.N2, gz = (z0 + pz) % p.N3;
                const long long ik = gx + (long long)p.N1 * (gy + (long long)p.N2 * gz);
                sW[k * WST + m] = (m0 + m < norb) ? load_out_weight(p, ik * p.sWk + (long long)n * p.sWn, m0 + m) : 0.0f;
            }
        } else {                   // k contiguous (SoA): lane = k-point, its MB orbitals fetched together (index arithmetic
                                   // once per k-point, MB independent loads in flight; neighbouring lanes read neighbouring k)
            for (int k = lane; k < PK; k += 32) {
                const int px = k % PX, py = (k / PX) % PY, pz = k / (PX * PY);
                const int gx = (x0 + px) % p.N1, gy = (y0 + py) % p.N2, gz = (z0 + pz) % p.N3;
                const long long ik = gx + (long long)p.N1 * (gy + (long long)p.N2 * gz);
                const long long wbase = ik * p.sWk + (long long)n * p.sWn;
                float v[MB];
#pragma unroll
                for (int m = 0; m < MB; m++) v[m] = (m0 + m < norb) ? load_out_weight(p, wbase, m0 + m) : 0.0f;
#pragma unroll
                for (int m = 0; m < MB; m++) sW[k * WST + m] = v[m];
            }
        }
        __syncwarp();

        // ---- A2/A3 (+ Eq. 14/15 constants): lane = (tetrahedron, band) record: sort, window, step histogram
        int lmin = 0x7fffffff, lmax = -1;
#pragma unroll 1
        for (int wd = 0; wd < NWORD; ++wd) {
            const int t = wd * 32 + lane;
            uint32_t rng = 0;   // i1 = i4 = 0: empty window
            float e0 = 0.f, e1 = 0.f, e2 = 0.f, e3 = 0.f;
            unsigned c0 = 0, c1 = 0, c2 = 0, c3 = 0;
            if (t < NTB) {
                const int tet = t / NC, cube = t - tet * NC;
                const int cx = cube % TX, cy = (cube / TX) % TY, cz = cube / (TX * TY);
                const bool valid = (x0 + cx < p.N1) && (y0 + cy < p.N2) && (z0 + cz < p.z_hi);
                const int cbase = cx + PX * (cy + PY * cz);
                {
                    const int a0 = kTableI[tet][0], a1 = kTableI[tet][1], a2 = kTableI[tet][2], a3 = kTableI[tet][3];
                    c0 = cbase + (a0 & 1) + PX * (((a0 >> 1) & 1) + PY * (a0 >> 2));
                    c1 = cbase + (a1 & 1) + PX * (((a1 >> 1) & 1) + PY * (a1 >> 2));
                    c2 = cbase + (a2 & 1) + PX * (((a2 >> 1) & 1) + PY * (a2 >> 2));
                    c3 = cbase + (a3 & 1) + PX * (((a3 >> 1) & 1) + PY * (a3 >> 2));
                }
                e0 = sE[c0]; e1 = sE[c1]; e2 = sE[c2]; e3 = sE[c3];
                TDOS_CSWAP(e0, e1, c0, c1);
                TDOS_CSWAP(e2, e3, c2, c3);
                TDOS_CSWAP(e0, e2, c0, c2);
                TDOS_CSWAP(e1, e3, c1, c3);
                TDOS_CSWAP(e1, e2, c1, c2);
                c0 *= WST; c1 *= WST; c2 *= WST; c3 *= WST;   // float offsets into sW
                if (valid) {
                    int i1, i4;   // first omega > E1; first omega >= E4, and > E1 (test order G10)
                    locate_window(om_loc, nE, om0, inv_dom, e0, e3, i1, i4);
                    rng = (uint32_t)i1 | ((uint32_t)i4 << 16);
                    if (mb == 0) {   // work counters (exact integers; bench.py's flop count uses them)
                        cnt_tb += 1;
                        cnt_ev += (unsigned)(i4 - i1);
                    }
                    if (i1 < i4) {
                        lmin = min(lmin, i1);
                        lmax = max(lmax, i4 - 1);
                    }
                    // Eq. 15 (A6): from the first omega >= E4 on, every corner carries the constant
                    // V: one add of sum_l b_l into the
                    // step histogram at bin i4 (all fp32 sums stay sums of non-negative terms)
                    if (i4 < nE) {
                        float b0[MB], b1[MB], b2[MB], b3[MB];
                        load_b<MB>(sW + c0, b0);
                        load_b<MB>(sW + c1, b1);
                        load_b<MB>(sW + c2, b2);
                        load_b<MB>(sW + c3, b3);
                        part_t* dst = part + (size_t)i4 * 3 * norb + 2 * norb + m0;
                        if constexpr (ACC64) {
#pragma unroll
                            for (int m = 0; m < MB; m++)
                                if (m0 + m < norb)
                                    red_add_f64(dst + m, ((double)b0[m] + (double)b1[m]) + ((double)b2[m] + (double)b3[m]));
                        } else if (vec4) {
                            if constexpr (MB % 4 == 0) {
#pragma unroll
                                for (int m4 = 0; m4 < MB; m4 += 4)
                                    if (m0 + m4 < norb)
                                        red_add4(dst + m4, (b0[m4] + b1[m4]) + (b2[m4] + b3[m4]),
                                                 (b0[m4 + 1] + b1[m4 + 1]) + (b2[m4 + 1] + b3[m4 + 1]),
                                                 (b0[m4 + 2] + b1[m4 + 2]) + (b2[m4 + 2] + b3[m4 + 2]),
                                                 (b0[m4 + 3] + b1[m4 + 3]) + (b2[m4 + 3] + b3[m4 + 3]));
                            }
                        } else {
#pragma unroll
                            for (int m = 0; m < MB; m++)
                                if (m0 + m < norb) red_add(dst + m, (b0[m] + b1[m]) + (b2[m] + b3[m]));
                        }
                    }
                }
            }
            sEs[t] = make_float4(e0, e1, e2, e3);
            sCs[t] = make_uint2(c0 | (c1 << 16), c2 | (c3 << 16));
            sRng[t] = rng;
        }
        lmin = __reduce_min_sync(FULL, lmin);
        lmax = __reduce_max_sync(FULL, lmax);
        __syncwarp();

        // ---- passes of PASS bins over the tile's energy span
#pragma unroll 1
        for (int pb = lmin; pb <= lmax; pb += PASS) {
            const int pe = pb + PASS;
            // -- which records overlap which chunk: bm[c][wd] bit j <=> record 32*wd+j has bins in chunk c
            int mycnt = 0;          // lane c: entries of chunk c
            uint32_t mywm = 0;      // lane c: non-empty words of chunk c
#pragma unroll 1
            for (int wd = 0; wd < NWORD; ++wd) {
                const uint32_t rr = sRng[wd * 32 + lane];
                const int i1 = (int)(rr & 0xffffu), i4 = (int)(rr >> 16);
                const bool has = (i1 < i4) && (i4 > pb) && (i1 < pe);
                int c1 = NCH, c2 = -1;
                if (has) {
                    c1 = (max(i1, pb) - pb) / CH;
                    c2 = (min(i4, pe) - 1 - pb) / CH;
                }
                const int cmin = __reduce_min_sync(FULL, c1);
                const int cmax = __reduce_max_sync(FULL, c2);
                uint32_t myword = 0;
                for (int c = cmin; c <= cmax; ++c) {
                    const uint32_t b = __ballot_sync(FULL, c1 <= c && c <= c2);
                    if (lane == c) myword = b;
                }
                sBm[lane * BST + wd] = myword;
                mycnt += __popc(myword);
                mywm |= (myword != 0u) ? (1u << wd) : 0u;
            }
            // -- exclusive prefix over chunks: the pass's (record, chunk) entries as one flat list
            int incl = mycnt;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int v = __shfl_up_sync(FULL, incl, d);
                if (lane >= d) incl += v;
            }
            const int off = incl - mycnt;
            const int T = __shfl_sync(FULL, incl, 31);
            sOff[lane] = off;
            sWm[lane] = mywm;
            __syncwarp();
            if (T == 0) continue;

            // -- even split of the flat list over the NG groups: group g takes entries [g*q, g*q + rem)
            const int q = (T + NG - 1) / NG;
            const int start = g * q;
            int rem = min(max(T - start, 0), q);
            const bool worked = rem > 0;
            int c = 0;
#pragma unroll
            for (int gg = 0; gg < NG; ++gg) {
                const uint32_t b = __ballot_sync(FULL, off <= gg * q);   // monotone: bits 0..c*
                if (gg == g) c = 31 - __clz(b);
            }
            int w = 0;
            uint32_t m = 0, wm = 0;
            if (worked) {   // position on entry `start`: skip whole words, then single records
                int skip = start - sOff[c];
                wm = sWm[c];
                for (;;) {
                    w = __ffs(wm) - 1;
                    wm &= wm - 1;
                    m = sBm[c * BST + w];
                    const int pc = __popc(m);
                    if (skip < pc) break;
                    skip -= pc;
                }
                for (; skip > 0; --skip) m &= m - 1;
            }
            int bin0 = pb + c * CH + 2 * gl;
            f2 om = make_float2((bin0 < nE) ? __ldg(omega + bin0) : qnan, (bin0 + 1 < nE) ? __ldg(omega + bin0 + 1) : qnan);

            typename std::conditional<ACC64, Acc64<MB>, Acc<MB>>::type acc;
            acc.zero();

            // -- A4-A6: every group walks its share of the list; lanes own bins
#pragma unroll 1
            for (int step = 0; step < q; ++step) {
                if (rem > 0) {
                    if (m == 0) {   // next non-empty word, possibly of the next chunk (uniform within the group)
                        while (wm == 0) {
                            acc.flush(part, bin0, nE, norb, m0, vec4);
                            ++c;
                            bin0 += CH;
                            om = make_float2((bin0 < nE) ? __ldg(omega + bin0) : qnan,
                                             (bin0 + 1 < nE) ? __ldg(omega + bin0 + 1) : qnan);
                            wm = sWm[c];
                        }
                        w = __ffs(wm) - 1;
                        wm &= wm - 1;
                        m = sBm[c * BST + w];
                    }
                    const int t = w * 32 + __ffs(m) - 1;
                    m &= m - 1;
                    --rem;

                    const float4 es = sEs[t];
                    const uint2 cs = sCs[t];
                    const unsigned cc[4] = {cs.x & 0xffffu, cs.x >> 16, cs.y & 0xffffu, cs.y >> 16};
                    bool done = false;
                    if constexpr (ACC64) {
                        if (p.w64) {   // TDOS_ACC_FP64_ALL: the weights themselves in double precision
                            double wa[4], da[4], wb[4], db[4];
                            corner_weights_f64((double)es.x, (double)es.y, (double)es.z, (double)es.w, (double)om.x, wa, da);
                            corner_weights_f64((double)es.x, (double)es.y, (double)es.z, (double)es.w, (double)om.y, wb, db);
                            const double w2[4][2] = {{wa[0], wb[0]}, {wa[1], wb[1]}, {wa[2], wb[2]}, {wa[3], wb[3]}};
                            const double d2[4][2] = {{da[0], db[0]}, {da[1], db[1]}, {da[2], db[2]}, {da[3], db[3]}};
                            acc.project64(sW, cc, w2, d2);
                            done = true;
                        }
                    }
                    if (!done) {
                        f2 wv[4], dw[4];
                        corner_weights_x2(es.x, es.y, es.z, es.w, om, wv, dw);
                        acc.project(sW, cc, wv, dw);
                    }
                }
            }
            if (worked) acc.flush(part, bin0, nE, norb, m0, vec4);
            __syncwarp();   // the next pass rewrites the bitmaps
        }
        __syncwarp();   // the next item rewrites the slice
    }

    cnt_tb = __reduce_add_sync(FULL, (unsigned)cnt_tb);   // per warp < 2^32
    unsigned long long ev = cnt_ev;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) ev += __shfl_xor_sync(FULL, ev, d);
    if (lane == 0 && (cnt_tb | ev)) {
        atomicAdd(p.counters + 0, cnt_tb);
        atomicAdd(p.counters + 1, ev);
    }
}

// Window statistics of a sample of the slab's cubes (A2/A3 only): est[0] += bins with E1 < omega < E4, est[1] += 1 per
// (tetrahedron, band).  The main kernels enqueued behind it read the two sums and the one that suits the windows
// runs (wanted_generation); no host round trip.
struct EstimateParams {
    const float* E;
    const float* omega;
    long long sEk, sEn;
    int N1, N2, N3, nb, nE;
    int z_lo, z_hi;
    int n_cubes;                 // cubes sampled, spread evenly over the slab
    unsigned long long* est;
};

__global__ void __launch_bounds__(256) tdos_estimate(const EstimateParams p) {
    const float* __restrict__ omega = p.omega;
    const float om0 = __ldg(omega);
    float inv_dom = 0.0f;
    if (p.nE > 1) {
        const float span = __ldg(omega + p.nE - 1) - om0;
        if (span > 0.0f) inv_dom = (float)(p.nE - 1) / span;
    }
    const long long slab = (long long)p.N1 * p.N2 * (p.z_hi - p.z_lo);
    const long long total = (long long)p.n_cubes * 6 * p.nb;
    unsigned long long bins = 0, cnt = 0;
    for (long long j = blockIdx.x * (long long)blockDim.x + threadIdx.x; j < total; j += (long long)gridDim.x * blockDim.x) {
        const int n = (int)(j % p.nb);
        const int tet = (int)((j / p.nb) % 6);
        const long long s = j / ((long long)p.nb * 6);
        const long long cube = (slab * s) / p.n_cubes;   // evenly spread
        const int ix = (int)(cube % p.N1), iy = (int)((cube / p.N1) % p.N2), iz = p.z_lo + (int)(cube / ((long long)p.N1 * p.N2));
        float emin = 3.0e38f, emax = -3.0e38f;
#pragma unroll
        for (int l = 0; l < 4; l++) {
            const int a = kTableI[tet][l];
            int gx = ix + (a & 1), gy = iy + ((a >> 1) & 1), gz = iz + (a >> 2);
            if (gx >= p.N1) gx -= p.N1;
            if (gy >= p.N2) gy -= p.N2;
            if (gz >= p.N3) gz -= p.N3;
            const long long ik = gx + (long long)p.N1 * (gy + (long long)p.N2 * gz);
            const float e = __ldg(p.E + ik * p.sEk + (long long)n * p.sEn);
            emin = fminf(emin, e);
            emax = fmaxf(emax, e);
        }
        const int i1 = locate_bin<true>(omega, p.nE, om0, inv_dom, emin);
        const int i4 = (emax > emin) ? locate_bin<false>(omega, p.nE, om0, inv_dom, emax) : i1;
        bins += (unsigned)(i4 - i1);
        cnt += 1;
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        bins += __shfl_xor_sync(0xffffffffu, bins, d);
        cnt += __shfl_xor_sync(0xffffffffu, cnt, d);
    }
    if ((threadIdx.x & 31) == 0 && cnt) {
        atomicAdd(p.est + 0, bins);
        atomicAdd(p.est + 1, cnt);
    }
}

// A7a: sum the block partials in fp64.  out[3][norb][nE] from per-block rows [nE][ D(norb) | T(norb) | S(norb) ].
__global__ void __launch_bounds__(256) tdos_merge(const float* __restrict__ partial, int nblk, int norb, int nE, int nEp,
                                                  double* __restrict__ out) {
    const size_t n = (size_t)3 * norb * nE, bstride = (size_t)3 * norb * nEp;
    for (size_t j = blockIdx.x * (size_t)blockDim.x + threadIdx.x; j < n; j += (size_t)gridDim.x * blockDim.x) {
        double s = 0.0;
        for (int c = 0; c < nblk; c++) s += (double)partial[(size_t)c * bstride + j];
        const size_t i = j / (3 * norb), qm = j - i * (3 * norb);
        out[qm * nE + i] = s;
    }
}

// A7a for fp64 partials
__global__ void __launch_bounds__(256) tdos_merge64(const double* __restrict__ partial, int nblk, int norb, int nE, int nEp,
                                                    double* __restrict__ out) {
    const size_t n = (size_t)3 * norb * nE, bstride = (size_t)3 * norb * nEp;
    for (size_t j = blockIdx.x * (size_t)blockDim.x + threadIdx.x; j < n; j += (size_t)gridDim.x * blockDim.x) {
        double s = 0.0;
        for (int c = 0; c < nblk; c++) s += partial[(size_t)c * bstride + j];
        const size_t i = j / (3 * norb), qm = j - i * (3 * norb);
        out[qm * nE + i] = s;
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
