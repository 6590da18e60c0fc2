/*
 * tetrados.h -- C ABI of libtetrados: linear-tetrahedron density of states on one B200.
 *
 * The library computes, for band energies E_n(k) and orbital weights
 * b_{n,m}(k) = |a_n^m(k)|^2 given on a periodic N1 x N2 x N3 k-grid,
 *
 *     DOS_m(w) = (1/V_G) sum_n int d^3k b_{n,m}(k) delta(w - E_n(k))      PAPER.md Eq. 4  (:52)
 *     N_m(w)   = (1/V_G) sum_n int d^3k b_{n,m}(k) Theta(w - E_n(k))      PAPER.md Eq. 2-3 (:43-48)
 *
 * by the linear tetrahedron method of arxiv 1710.10789: every cube of the grid is split into
 * the six tetrahedra of Table I, the four corner energies of each
 * (tetrahedron, band) are sorted, the corner weights w_l(w) and dw_l/dw of
 * Eq. 11-15 are evaluated and contracted with the corner orbital weights
 * (Eq. 8, :91) and summed over tetrahedra and bands (Eq. 9, :96).  Everything runs in CUDA
 * kernels for sm_100a; there is no CPU fallback.
 *
 * Conventions (part of the ABI)
 *   k-point index   ik = ix + N1*(iy + N2*iz), ix fastest; k = (ix/N1, iy/N2, iz/N3) in units of the
 *                   reciprocal lattice vectors; the grid is periodic (index N_d wraps to 0), so there
 *                   are N1*N2*N3 cubes.  The cube at ik has its corner 1 there; corner label c=1..8 of
 *                   Table I sits at offset (dx,dy,dz) = bits 0,1,2 of (c-1)   (reading G7).
 *   normalisation   V_T/V_G = 1/(6 N1 N2 N3); no spin factor.  N_m(w -> inf) = (1/nk) sum_k sum_n b.
 *   intervals       half-open, tested in the order  w <= E1, w < E2, w < E3, w < E4, else  (reading G10).
 *   precision       fp32 inputs, fp32 arithmetic for the weights, block-local fp32
 *                   partial sums, fp64 merge across blocks and fp64 prefix sum for N; fp32 outputs
 *                   (tdos_plan_set_accumulation widens every sum to fp64).
 *   reproducibility results are reproducible to rounding, NOT bit for bit: the block partials are built with
 *                   fire-and-forget reductions in L2 (red.global.add) in arrival order and work items are drawn
 *                   from a global counter, so the order of the fp32 additions differs from run to run
 *                   (differences ~1e-7 relative, two orders below the tolerances of BASELINE.json).
 *   NaN/Inf in E or W are not detected: results are then undefined.
 *   omega           must be strictly increasing.  Host mode checks it (TDOS_EINVAL); DEVICE mode does NOT -- the
 *                   array lives on the device and the call only enqueues work -- a non-monotonic device array
 *                   gives undefined results (no fault: bin indices are clamped to [0, nE]).
 *
 * Kernels: tdos_main5 (one record per interval of Eq. 12-14; blocks of 8 orbitals: norb >= 5 and norb % 4 == 0) and
 * tdos_main (one record per tetrahedron; any norb).  A plan that qualifies for tdos_main5 carries both: every call
 * first enqueues tdos_estimate, which samples the windows (E1, E4) of 2048 cubes on the device, then both main
 * kernels; the one that suits the windows runs (tdos_main below 7 energies per window on average, tdos_main5
 * above), the other returns at once.  Nothing is decided on the host and nothing is remembered between calls.
 * (In TDOS_HOST mode the sample is taken from the first staged z-slab, the only planes on the device at that time.)
 * Environment variables read at plan creation, for tests and experiments only: TDOS_KERNEL=3|5 forces one kernel,
 * TDOS_TILE=<index> forces one of the compiled tile shapes (generation 5: 0 = 4x4x2, 1 = 2x2x8 cubes per warp;
 * generation 3 on blocks of 8 orbitals: 0 = 2-lane groups, 1 and 2 = the short-window kernels).  A library built with
 * -DTDOS_EXPERIMENTS carries more shapes and reads TDOS_BLOCKS_PER_SM (DESIGN.md section 4 and the experiments logs).
 *
 * Ownership: the caller owns every array; the library never frees them and does not retain them
 * past the call (device mode: past completion of the work queued on `stream`).  A plan owns all
 * scratch (block partials, staging buffers, its side stream), shared by all its calls: calls are executed one after the
 * other even when issued on different streams (a call on another stream than the previous one first waits, on the
 * device, for that one's end).  A plan must not be used from two host threads at the same time.  Inputs are never
 * written.  CUDA graphs: a TDOS_DEVICE call (tetra_dos, _select, _complex, _partial, _partial_slab, _finalize) whose
 * stream is being captured is recorded into the graph -- memsets and kernels only; the plan's ordering and timing
 * events are left out, so tdos_kernel_ms does not see it and a replay is ordered against other calls on the plan only
 * by what the caller orders: do not run a replay concurrently with another call on the same plan.  The call captured
 * first on a plan should not be the plan's very first call (the first call of a kernel loads it).  Every entry point runs on the plan's device and restores the caller's current device before it returns.
 *
 * Errors: every function returns 0 (TDOS_OK) or a negative code; nothing throws, exits or prints.
 * On error the outputs are untouched (host mode) / unspecified only if TDOS_ECUDA occurred mid-flight.
 */
#ifndef TETRADOS_H
#define TETRADOS_H

#ifdef __cplusplus
extern "C" {
#endif

#define TDOS_OK       0
#define TDOS_EINVAL  -1   /* bad argument: NULL where not allowed, N_d < 1, nb/norb/nE < 1, nE > nE_max,
                             nE > TDOS_MAX_NE, omega not strictly increasing, W == NULL with norb != 1,
                             bad layout / memspace / slab range                                       */
#define TDOS_ENOMEM  -2   /* host or device allocation failed                                          */
#define TDOS_ECUDA   -3   /* a CUDA call failed; see tdos_last_cuda_error()                            */
#define TDOS_EARCH   -4   /* the selected device is not compute capability 10.x (sm_100)               */
#define TDOS_ESIZE   -5   /* tetra_dos_static only: the problem needs more scratch than the library's built-in
                             buffer holds (norb * nE above TDOS_STATIC_MAX_CELLS); use a plan instead  */

#define TDOS_AOS 0        /* E[ik][n],  W[ik][n][m]   -- what a CPU code usually holds                  */
#define TDOS_SOA 1        /* E[n][ik],  W[n][m][ik]   -- k fastest                                      */

#define TDOS_DEVICE 0     /* E, W, omega, dos, nos are device pointers (on the plan's device)           */
#define TDOS_HOST   1     /* they are host pointers (pinned recommended); H2D / D2H done by the library */

#define TDOS_MAX_NE 65534 /* energies per call (bin indices are kept in 16 bits inside the kernel)      */

typedef struct tdos_plan tdos_plan;   /* opaque */

/* Library version (major*100 + minor). */
int tdos_version(void);

/* Static, never-freed description of an error code. */
const char* tdos_strerror(int code);

/* Text of the last CUDA error seen by the calling thread ("" if none).  Valid until the next
 * failing call on this thread. */
const char* tdos_last_cuda_error(void);

/*
 * Create a plan for grids of nk[0] x nk[1] x nk[2] k-points, nb bands, norb orbitals and up to
 * nE_max energies on CUDA device `device`.  Allocates all device scratch:
 * per-block partial histograms (3 * (norb + 1 rounded up to 4) * (nE_max + 3) floats per resident block, 148 blocks on
 * a B200) and the fp64 merge buffer.  *out is set only on success.
 */
int tdos_plan_create(tdos_plan** out, int device, const int nk[3], int nb, int norb, int nE_max);

/*
 * Precision of the accumulation (Sec. III.B: single precision throughout, "one can in principle switch
 * to double precision").  TDOS_ACC_FP32 (default): fp32 sums in registers and block partials, fp64 merge and prefix sum.
 * TDOS_ACC_FP64: the corner weights are still evaluated in single precision, but every sum taken after them (registers,
 * block partials, the Eq.-15 step histogram, merge, prefix sum) is fp64; slower (about 3x on config 4), results agree
 * with the fp64 oracle to ~1e-7 relative instead of ~1e-6.  Allocates a second, fp64 set of block
 * partials the first time the mode is chosen (TDOS_ENOMEM if that fails); waits for the plan's last call.
 * TDOS_ACC_FP64_ALL: the corner weights of Eq. 11-14 are evaluated in double precision as well (true divisions instead
 * of rcp.approx), so the whole path after the fp32 inputs is fp64; the fp64 shares of tetra_dos_partial then agree
 * with the fp64 oracle to ~1e-12 relative (the fp32 outputs of tetra_dos still round to 6e-8).  Slowest mode.
 */
#define TDOS_ACC_FP32 0
#define TDOS_ACC_FP64 1
#define TDOS_ACC_FP64_ALL 2
int tdos_plan_set_accumulation(tdos_plan* p, int mode);

/* Free a plan and everything it owns.  NULL is a no-op.  Synchronises the plan's streams first. */
int tdos_plan_destroy(tdos_plan* p);

/*
 * The hot path: DOS_m(omega_i) and N_m(omega_i) for all orbitals m and all nE energies.
 *
 *  E       band energies, nk*nb floats in `layout`
 *  W       orbital weights |a_n^m(k)|^2, nk*nb*norb floats in `layout`;
 *          NULL means W == 1 and requires norb == 1 (total DOS, X = 1)
 *  omega   nE strictly increasing energies.  A (nearly) uniform grid is located by direct
 *          index computation plus an exact fix-up; any other increasing grid is still handled
 *          exactly, only slower.
 *  dos     out [norb][nE], overwritten
 *  nos     out [norb][nE], overwritten; may be NULL
 *  memspace TDOS_DEVICE: all five pointers are device pointers; the call only enqueues work on
 *          `cuda_stream` (a cudaStream_t, NULL = legacy default stream) and returns; no host synchronisation.
 *          TDOS_HOST: all five are host pointers; inputs are staged to the device in z-slabs on the
 *          plan's side stream, overlapped with the kernels, and the call returns after the results
 *          are in `dos` / `nos` (`cuda_stream` is ignored).
 */
int tetra_dos(tdos_plan* p, const float* E, const float* W, int layout, const float* omega, int nE,
              float* dos, float* nos, int memspace, void* cuda_stream);

/*
 * The same with the eigenvector elements themselves (Eq. 1-3, :37-48; the paper's kernel takes real and
 * imaginary parts, :263): A holds nk*nb*norb complex numbers as (re, im) float pairs in `layout`
 * (TDOS_AOS: A[ik][n][m][2], TDOS_SOA: A[n][m][ik][2]); the kernels form b = re^2 + im^2 while staging a tile.
 * A must not be NULL.  Everything else as tetra_dos.
 */
int tetra_dos_complex(tdos_plan* p, const float* E, const float* A, int layout, const float* omega, int nE,
                      float* dos, float* nos, int memspace, void* cuda_stream);

/*
 * Orbital selection plus total ("the five Fe 3d orbitals ... and the total density of states" of an
 * 8-orbital model; reading G15: total = sum over ALL orbitals).  Rows of dos / nos:
 *     j < nsel : orbital orbitals[j] (0-based, each < norb and <= 32767, any order, repeats allowed),
 *     j = nsel : sum over all norb orbitals, present if want_total != 0.
 * dos, nos are [nsel + (want_total != 0)][nE]; nsel <= 32, at most norb + 1 rows; nsel = 0 with want_total gives the
 * total alone.  W must not be NULL; `orbitals` is a HOST array in both memory spaces.  Everything else as tetra_dos.
 * The selection is applied while a tile is staged, so only the rows asked for are projected and accumulated.
 */
int tetra_dos_select(tdos_plan* p, const float* E, const float* W, int layout, const float* omega, int nE,
                     const int* orbitals, int nsel, int want_total, float* dos, float* nos, int memspace,
                     void* cuda_stream);

/*
 * The step before the path, on the device (Eq. 1, :37-39: the tight-binding Hamiltonian H(k) is "diagonalised
 * to obtain band energies E_n(k) and eigenvector elements a_n^m(k)"; :289: the best case is input that already
 * resides in GPU memory): batched Hermitian eigensolver for plans with nb == norb <= 16 (the paper's model: 8; "16
 * orbitals correspond to the largest models ... currently considered", :269).
 *   H  in  device, nk*nb*nb complex numbers as (re, im) float pairs, H[ik][i][j] row-major, Hermitian: only the upper
 *      triangle (j >= i) and the real part of the diagonal are read, the rest is taken as its conjugate
 *   E  out device [nk][nb], ascending per k-point                                     (TDOS_AOS layout of tetra_dos)
 *   A  out device [nk][nb][nb][2]: A[ik][n][m] = a_n^m(k), component m of eigenvector n (TDOS_AOS layout of
 *      tetra_dos_complex), normalised, phase arbitrary
 * so that  tetra_eigh(p, H, E, A, s); tetra_dos_complex(p, E, A, TDOS_AOS, ...)  goes from H(k) to the DOS without a
 * host round trip.  Cyclic Jacobi, fp64 arithmetic like the host LAPACK call it replaces (sweeps until the off-diagonal
 * norm is below 1e-12 of the matrix norm, at most 10; 14 for orders above 8), results rounded to the fp32 arrays the
 * path consumes; 8 lanes per matrix up to order 8, 16 lanes above.  Asynchronous on `cuda_stream`.  TDOS_EINVAL if nb != norb or nb > 16.
 */
int tetra_eigh(tdos_plan* p, const float* H, float* E, float* A, void* cuda_stream);

/*
 * Multi-GPU building blocks (device pointers only).
 * tetra_dos_partial: the additive share of the cubes with z_lo <= iz < z_hi, as raw fp64 sums
 *   part[3][norb][nE]  (0: sum b*dw/V, 1: sum b*w/V over E1 < omega < E4, 2: Eq.-15 step histogram / V at the first omega >= E4),
 *   overwritten.  E and W must hold the whole grid (the kernel reads planes z_lo .. z_hi, wrapping).
 * tetra_dos_finalize: dos = V*part[0]; nos = V*(part[1] + inclusive prefix sum over omega of part[2]).
 * A sum of the `part` arrays of disjoint slabs covering 0..N3 (e.g. an all-reduce) followed by
 * tetra_dos_finalize equals tetra_dos.
 */
int tetra_dos_partial(tdos_plan* p, const float* E, const float* W, int layout, const float* omega,
                      int nE, int z_lo, int z_hi, double* part, void* cuda_stream);
int tetra_dos_finalize(tdos_plan* p, const double* part, int nE, float* dos, float* nos,
                       void* cuda_stream);
/*
 * tetra_dos_partial for a GPU that holds only its own part of the grid ("each GPU holding its slab's
 * k-planes plus one halo plane"): E and W hold the z_hi - z_lo + 1 k-planes z_lo, z_lo + 1, ..., z_hi of
 * the grid in this order -- the last one is the halo, i.e. plane 0 again when z_hi == N3 -- and nothing else:
 *     TDOS_AOS: E[kl][n], W[kl][n][m];   TDOS_SOA: E[n][kl], W[n][m][kl];   kl = ix + N1*(iy + N2*(iz - z_lo)),
 * (N1*N2*(z_hi - z_lo + 1) k-points).  Requires z_lo < z_hi.  `part` and everything else as tetra_dos_partial; the two
 * calls give the same share for the same slab.
 */
int tetra_dos_partial_slab(tdos_plan* p, const float* E, const float* W, int layout, const float* omega,
                           int nE, int z_lo, int z_hi, double* part, void* cuda_stream);

/*
 * Generic tetrahedron integration weights (Eq. 5-7, :58-71): for nW energies (device array, any order)
 *     wk[e][n][ik]  = sum over the tetrahedra with corner ik of w_{n,l}(energies[e])        (Eq. 11-15)
 *     dwk[e][n][ik] = the same with dw/dE (may be NULL),
 * both [nW][nb][nk] floats on the device, k fastest, overwritten, normalised so that
 * <X>(E) = sum_n sum_ik X_n(k_ik) wk[e][n][ik] (Eq. 7); X = 1 gives the integrated DOS, X = b_{n,m} gives N_m.
 * E in `layout` as for tetra_dos; the plan's norb is not used.  Asynchronous on `cuda_stream`.
 */
int tetra_weights(tdos_plan* p, const float* E, int layout, const float* energies, int nW, float* wk, float* dwk,
                  void* cuda_stream);

/*
 * One-shot convenience matching the paper's "called from a CPU code" scenario:
 * host pointers, AoS layout, cubic Nk^3 grid, omega_i = (float)(omega_min + i*(omega_max-omega_min)/(nE-1))
 * evaluated in double (endpoints inclusive).  Creates a plan on the current device,
 * runs, destroys it.
 */
int tetra_dos_simple(const float* E, const float* W, int Nk, int nb, int norb, float omega_min,
                     float omega_max, int nE, float* dos, float* nos);

/*
 * tetra_dos for callers that are not allowed to allocate device memory.
 *
 * Who that is: code that runs where cudaMalloc is off limits -- a plug-in inside a host program (a DFT/DMFT driver,
 * say) that has sized its own memory pools to fill the GPU and requires every byte of device memory to come from
 * them, so a cudaMalloc either fails or breaks the host's accounting; and a self-consistency or real-time loop that
 * cannot afford the device-wide synchronisation that cudaMalloc / cudaFree imply in the middle of its pipeline.
 * A tdos_plan is no use to them: creating one allocates its block partials, merge buffer, streams and events.
 *
 * This call needs no plan and allocates nothing -- no cudaMalloc, no cudaFree, no stream, no event.  The scratch every
 * DOS call needs (block-partial histograms, the fp64 merge buffer, the work counters) lives in an array that is built
 * into the library image: TDOS_STATIC_SCRATCH_BYTES (about 16.8 MB) of device memory on EVERY GPU on which the
 * process loads the library, held until the process exits whether or not this function is ever called.  The price
 * of a fixed buffer is a size limit:
 *
 *     norb * (nE rounded up to a multiple of 4)  <=  TDOS_STATIC_MAX_CELLS  (32768: e.g. 8 orbitals x 4096 energies,
 *                                                                            16 x 2048, 1 x 32768)
 *
 * Anything larger returns TDOS_ESIZE and touches nothing.  The fewer cells a call uses, the more thread blocks get a
 * private histogram (up to one per resident block; at the limit 42 blocks share the GPU), so small problems run at
 * plan speed and problems at the limit run slower than through a plan.
 *
 * Arguments as tetra_dos in TDOS_DEVICE mode: E, W (NULL = unit weights, needs norb == 1), omega, dos, nos (may be
 * NULL) are device pointers on the CURRENT device, which must be an sm_100 GPU (TDOS_EARCH otherwise); the grid shape,
 * nb and norb are passed directly since there is no plan; the work is enqueued on `cuda_stream` and the call returns
 * without waiting.  Only the one-record-per-tetrahedron kernel (tdos_main) is used; results agree with tetra_dos to
 * rounding (different summation order), not bit for bit.
 *
 * First call on a device: looks up the device address of the built-in buffer, sets the kernels' shared-memory limit
 * and queries their occupancy, and remembers all three for later calls (guarded by a mutex; later calls only check a
 * flag).  Make that first call per device outside any stream capture; it is also the call that may trigger the CUDA
 * runtime's own lazy loading of the kernels.
 *
 * All calls in a process share the one buffer per device.  Each call clears what it needs before it uses it, so
 * calls that follow each other on one stream (or are otherwise ordered on the GPU) are independent of each other's
 * sizes and contents.  Calls that can OVERLAP on the same GPU -- two streams, two host threads -- race on the buffer
 * and give wrong results without any error; ordering them is the caller's job.  Plans are unaffected: they use their
 * own scratch.
 */
#define TDOS_STATIC_MAX_CELLS     32768
#define TDOS_STATIC_SCRATCH_BYTES (256 + 3 * TDOS_STATIC_MAX_CELLS * 8 + (16 << 20))
int tetra_dos_static(const int nk[3], int nb, int norb, const float* E, const float* W, int layout,
                     const float* omega, int nE, float* dos, float* nos, void* cuda_stream);

/*
 * Diagnostics used by bench.py (not part of the hot path).
 * tdos_plan_info: what[0] = resident blocks of the main kernel, [1] = threads per block,
 *   [2] = dynamic shared memory per block (bytes), [3] = work items of the last call,
 *   [4] = kernel launches of the last tetra_dos / tetra_dos_partial+finalize call,
 *   [5..7] = tile extent in cubes (x, y, z).
 * tdos_last_counters: exact work counters of the last tetra_dos / tetra_dos_partial call, counted by
 *   the main kernel: cnt[0] = n_tb = (tetrahedron, band) pairs processed, cnt[1] = n_eval = number of
 *   (tetrahedron, band, omega_i) with E1 < omega_i < E4, i.e. evaluations of Eq. 12-14 the method
 *   needs; cnt[2] = how many of them fall in the middle interval E2 <= omega_i < E3
 *   (Eq. 13; -1 if the kernel that ran does not count it), cnt[3] = generation of the main kernel that ran
 *   (3 = tdos_main, 5 = tdos_main5; for a plan carrying both: what the device decided for that call).
 *   Synchronises the call's stream.
 * tdos_kernel_ms: mean device time of the main kernel and of the merge+finalize kernels over the
 *   last `ncalls` (1..64) device-mode tetra_dos calls on this plan, from CUDA events the library records
 *   on each call's stream around its own launches (waits for those calls to finish); the "main kernel" bracket
 *   holds the scratch memsets, tdos_estimate and both main kernels of a plan that carries two.
 *   tdos_last_kernel_ms is tdos_kernel_ms with ncalls = 1.
 * tdos_fp32_fma_probe: runs a register-resident FFMA chain on every SM of the plan's device and
 *   returns the achieved FP32 rate in TFLOP/s (2 flops per FMA lane) in *tflops.
 */
int tdos_plan_info(const tdos_plan* p, long long what[8]);
int tdos_last_counters(tdos_plan* p, long long cnt[4]);
int tdos_kernel_ms(tdos_plan* p, int ncalls, float* main_ms, float* merge_ms);
int tdos_last_kernel_ms(tdos_plan* p, float* main_ms, float* merge_ms);
int tdos_fp32_fma_probe(tdos_plan* p, int packed, double* tflops);

#ifdef __cplusplus
}
#endif
#endif /* TETRADOS_H */
