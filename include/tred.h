/*
 * tred.h -- C ABI of the B200-native TRED hot path (arxiv 2602.12052).
 *
 * "Segments in, per-pixel current waveforms out" (Fig. 1):
 *
 *   tred_drift            R/A/D of Fig. 1: attachment, drift, diffusion width
 *   tred_blockbin         block-sparse binned tensor: occupied-block list
 *   tred_effq             effective charge, Eq. (9)-(10)
 *   tred_convolve         interlaced FFT convolution, Eq. (12)/(14)
 *   tred_gather_waveforms overlap-add of block outputs on unique pixels
 *
 * Conventions
 *   - Every pointer named d_* is DEVICE memory, h_* is HOST memory.  All device buffers,
 *     workspaces included, are allocated by the caller and only borrowed; the library
 *     never allocates device memory and the stepwise calls never synchronise the host
 *     (exceptions: tred_prepare_response, once per response; tred_profile_end; and
 *     tred_simulate, which reads the device-side counts once per event to size what follows --
 *     it keeps 64 KB of pinned host memory per context for that).  Calls are enqueued on
 *     `stream` (a cudaStream_t passed as void*).
 *   - Results of data-dependent size use "capacity + device-side count": the count is
 *     written to device memory; entries beyond the capacity are not written.  The caller
 *     reads the count (its own synchronisation), re-allocates and calls again if needed.
 *   - Return value: TRED_OK or a negative tred_status.  TRED_ECUDA reports the CUDA error
 *     seen when the kernels were enqueued; asynchronous faults surface on the caller's
 *     next synchronisation.
 *   - Units: mm, microseconds, electrons.  Fine grid G: point (i,j,k)
 *     is the CENTRE of cuboid (i,j,k): x = origin_x + (i+1/2) h, h = pitch/sub,
 *     t = t_origin + (k+1/2) tick.  Pixel P = i div sub, sub-pixel phase j = i mod sub.
 *   - Block key (int64): (bt*NBx + bx)*NBy + by, time slab major; keys are sorted
 *     ascending.  Tile / slab-pixel key: (tb*npix_x + px)*npix_y + py.
 *   - Charge outside the grid and current outside the pixel plane / readout window are
 *     dropped (reading G13).
 *   - A context belongs to the CUDA device that was current in tred_create; a call made while
 *     another device is current returns TRED_EINVAL (several contexts, one per device, may live
 *     in one process).
 *   - There is no CPU fallback: without a CUDA device every compute call fails.
 */
#ifndef TRED_H
#define TRED_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum tred_status {
  TRED_OK = 0,
  TRED_EINVAL = -1,        /* bad argument or configuration                    */
  TRED_ECAP = -2,          /* caller-provided capacity / workspace too small   */
  TRED_ECUDA = -3,         /* CUDA runtime error (see tred_last_cuda_error)    */
  TRED_EUNSUPPORTED = -4   /* configuration outside what the kernels support   */
} tred_status;

/* Plain-data configuration, host memory, copied by tred_create. */
typedef struct tred_config {
  int32_t npix_x, npix_y;        /* pixel plane                                           */
  int32_t sub;                   /* S: sub-pixel factor (10)               */
  int32_t nticks;                /* readout window in ticks                               */
  double  pitch_mm, tick_us;
  double  origin_x_mm, origin_y_mm, t_origin_us;
  double  v_mm_us;               /* drift velocity                                        */
  double  lifetime_us;           /* electron lifetime tau                                 */
  double  DL_mm2_us, DT_mm2_us;  /* longitudinal / transverse diffusion coefficients      */
  double  sigma_min_xy_mm, sigma_min_t_us;   /* minimum diffusion scale   */
  double  nsigma;                /* half-width of the charge box in sigmas (reading G9)   */
  double  point_thresh;          /* point/line switch, PAPER.md:L148 (0.1)                */
  int32_t gl_n;                  /* Gauss-Legendre points per axis, 1..4                  */
  int32_t block[3];              /* Bx, By (fine-grid points), Bt (ticks): powers of two  */
  int32_t resp_half;             /* H: response covers (2H+1)^2 pixels                    */
  int32_t resp_nticks;           /* Tr: response length in ticks                          */
  int32_t effq_mode;             /* how tred_effq evaluates the charge density of Eq. (10):
                                    0 = factored line integral (default, see tred_effq),
                                    1 = closed form with erf per Gauss-Legendre node          */
  int32_t mac_mode;              /* spectrum multiply-accumulate of tred_convolve:
                                    0 = default: the best of the modes below this configuration
                                        supports, tried in the order 7, 6, 3, 2, 1
                                        (tred_last_mac_mode reports the one that ran),
                                    7 = tensor cores over row tiles with the sum over the offsets
                                        fused into the epilogue, on CTA pairs (tcgen05
                                        cta_group::2); operands split x = s (hi + lo), hi and lo
                                        fp16, s a power of two per row / per frequency; the three
                                        products hi*hi, lo*hi, hi*lo in fp16 with fp32
                                        accumulation; the forward FFT writes the split operands,
                                    6 = as 7 with fp32 spectra split in the kernel: hi*hi in tf32,
                                        the two corrections in bf16,
                                    5 = as 6 with all three products in tf32 (3xTF32),
                                    3 = as 5 on single CTAs,
                                    4 = as 5 with the mirror symmetry of the response
                                        (MPCP) spent on the product: sums and
                                        differences of mirror phase pairs, two products of half
                                        the size; if the response prepared last is not exactly
                                        mirror-symmetric the general product of mode 6 runs
                                        instead (never the fp16 path of mode 7) and
                                        tred_last_mac_mode reports 6,
                                    1 = fp32 FMA pipe, products written to memory,
                                    2 = tensor cores 3xTF32, products written to memory       */
  int32_t fft_mode;              /* forward transform of tred_convolve in mac_mode 7:
                                    0 = default: pruned DFT as a dense contraction on the tensor
                                        cores (tred_dft_h16.cu) where the shape allows it (S = 10;
                                        Bt a multiple of 32, <= 128; L with a divisor NC <= 256,
                                        NC a multiple of 32, L / NC >= 2; and half of the DFT
                                        matrix, L * Bt * 2 bytes, plus Bt * 512 bytes of operand
                                        tile and ~2 KB fit the opt-in shared memory of one CTA:
                                        L * Bt <= ~80 000 on B200), else as 1,
                                    1 = shared-memory / register FFT kernels                     */
} tred_config;

/* Sizes derived from a configuration (host-side helper, no device work). */
typedef struct tred_dims {
  int64_t NG[3];          /* fine-grid points (x, y, t)                                   */
  int64_t NB[3];          /* blocks per axis = ceil(NG/B)                                 */
  int32_t fft_len;        /* L: smallest 2^a 3^b (a >= 3) >= Bt + Tr - 1 (reading G20;
                             PAPER.md:L264 pads to a power of two)                        */
  int32_t out_len;        /* Bt + Tr - 1: ticks of one block's output                     */
  int32_t n_over;         /* ceil(out_len / Bt): tiles (Tt = Bt) one output spans         */
  int32_t n_freq;         /* L/2 complex spectrum slots (slot 0 packs DC and Nyquist)     */
  int32_t n_phase;        /* S*S sub-pixel phases                                         */
  int32_t n_off;          /* (2H+1)^2 pixel offsets of the response                       */
  int32_t n_off_pad;      /* n_off rounded up to a multiple of 8                          */
  int32_t pix_per_block;  /* max charge pixels met by one block: product over x, y of
                             floor((S - 1 + B - 1)/S) + 1                                 */
  int64_t rhat_floats;    /* floats of the response spectrum buffer (all layouts)         */
  int64_t block_floats;   /* Bx*By*Bt                                                     */
  int64_t conv_row_bytes; /* tred_convolve workspace bytes per charge pixel in flight     */
  int32_t dft_ticks;      /* Bt: rows of the DFT matrix kept with the response spectrum   */
} tred_dims;

typedef struct tred_ctx tred_ctx;   /* opaque, host memory */

int  tred_get_dims(const tred_config* cfg, tred_dims* out);
int  tred_create(const tred_config* cfg, tred_ctx** out);
void tred_destroy(tred_ctx* ctx);
const char* tred_strerror(int status);
const char* tred_last_cuda_error(void);
int  tred_abi_version(void);
/* The spectrum-product kernel (a tred_config.mac_mode value 1..7) the last tred_convolve on
 * this context launched; 0 before the first call.  A mode the configuration cannot run is
 * replaced as tred_config.mac_mode describes, never silently: this is where it shows. */
int  tred_last_mac_mode(const tred_ctx* ctx);

/* Number of floats / int32 per segment in the augmented SoA record (see tred_drift). */
#define TRED_AUG_NF 10
#define TRED_AUG_NI 8

/*
 * tred_drift -- PAPER.md:L41,L57 (A, D of Fig. 1); readings G6-G11, G14 in DESIGN.md.
 *   d_seg    [8][nseg] float32 SoA rows x0,y0,z0,x1,y1,z1,q,t0 (row stride = nseg);
 *            z = drift distance to the anode, q = electrons after recombination.
 *   d_augf   [TRED_AUG_NF][nseg] float32 out: p0x,p0y,p0t,p1x,p1y,p1t (segment ends in
 *            grid units relative to the bbox corner `lo`), sx,sy,st (sigma in grid units),
 *            Q' = q exp(-t_m/tau).
 *   d_augi   [TRED_AUG_NI][nseg] int32 out: lox,loy,lot,hix,hiy,hit (inclusive cuboid
 *            bounding box, may lie partly outside the grid), flag (1 = point-like),
 *            npair (number of blocks the clipped grid-point footprint meets).
 *   d_npairs int64 out: sum of npair (zeroed by the call).
 *   The integer outputs are computed in fp64, round-to-nearest, without FMA
 *   contraction, in the operation order DESIGN.md states: they are bit-exact.
 */
int tred_drift(tred_ctx* ctx, int64_t nseg, const float* d_seg,
               float* d_augf, int32_t* d_augi, int64_t* d_npairs, void* stream);

/*
 * tred_blockbin -- block-sparse binned tensor (readings G15,G16):
 * expands every segment into (block key, segment) pairs, radix-sorts them by key
 * (stable), run-length compacts the keys.  The payload [nblocks][Bx][By][Bt] is laid out
 * by this list and filled by tred_effq.
 *   cap_pairs   capacity of d_pair_seg (>= *d_npairs of tred_drift)
 *   d_keys      [cap_blocks] int64 out: sorted unique keys of the occupied blocks
 *   d_blk_off   [cap_blocks+1] int32 out: CSR offsets into d_pair_seg
 *   d_pair_seg  [cap_pairs] int32 out: segment ids grouped by block, ascending in a block
 *   d_slab_off  [NBt+1] int32 out: first block index of every time slab
 *   d_nblocks   int64 out: number of occupied blocks (may exceed cap_blocks: TRED_ECAP
 *               semantics, nothing beyond the capacity is written)
 *   d_work      workspace of at least tred_blockbin_work_bytes(nseg, cap_pairs) bytes
 */
size_t tred_blockbin_work_bytes(const tred_ctx* ctx, int64_t nseg, int64_t cap_pairs);
int tred_blockbin(tred_ctx* ctx, int64_t nseg, const int32_t* d_augi,
                  int64_t cap_pairs, int64_t cap_blocks,
                  int64_t* d_keys, int32_t* d_blk_off, int32_t* d_pair_seg,
                  int32_t* d_slab_off, int64_t* d_nblocks,
                  void* d_work, size_t work_bytes, void* stream);

/*
 * tred_effq -- effective charge, Eq. (9) with Eq. (10) / the point-like branch
 * (readings G1, G4, G5, G10).  One CTA per block tile, the tile
 * staged in shared memory, no atomics, fixed summation order.
 *   effq_mode 0: the charge density at a Gauss-Legendre node is the line integral that
 *     Eq. (10) is the closed form of, q = Q' int_0^1 prod_a N(r_a - p0_a - s d_a; sigma_a) ds,
 *     evaluated by an m-point Gauss-Legendre rule in s with m chosen per segment so that
 *     the relative error is < 1.5e-7 (below fp32 rounding of the result).  Every term is
 *     separable in (x, y, t), so the sums over the n^3 nodes and the trilinear
 *     coefficients u of Eq. (9) factor into three 1-D tables per segment.
 *     The tables of the segments a range of blocks refers to are built once, in d_work
 *     (a segment meets several blocks), and copied by the tile CTAs.
 *   effq_mode 1: Eq. (10) in closed form (exp, erf) at every node.
 *   d_payload [nblocks][Bx][By][Bt] float32 out (fully overwritten).
 *   d_work    workspace of tred_effq_work_bytes(nseg) bytes (less, or NULL, is allowed: the
 *             tables are then rebuilt by every CTA -- same values, slower).
 */
size_t tred_effq_work_bytes(const tred_ctx* ctx, int64_t nseg);
int tred_effq(tred_ctx* ctx, int64_t nseg, int64_t nblocks,
              const int64_t* d_keys, const int32_t* d_blk_off, const int32_t* d_pair_seg,
              const float* d_augf, const int32_t* d_augi,
              float* d_payload, void* d_work, size_t work_bytes, void* stream);

/*
 * tred_prepare_response -- FFT(R^j) of Eq. (14), computed once.
 *   d_resp [S][S][2H+1][2H+1][Tr] float32: R[jx][jy][kx+H][ky+H][tau] = current at tick
 *          tau on the pixel displaced by (kx,ky) from the pixel holding a unit charge at
 *          sub-pixel phase (jx,jy) (readings G3, G12).
 *   d_rhat [rhat_floats] float32 out: the spectrum in the layouts the kernels read
 *          (fp32 [f][phase][offset] complex, and the real-ified matrices
 *          [f][2*offset+c][2*phase+c'] split into tf32 hi / lo parts for the tensor cores,
 *          and the half-size matrices of a mirror-symmetric response).
 *   Dynamic range in mac_mode 7 (the default): the fp16 hi / lo parts of the spectrum share one
 *   power-of-two scale per frequency across all phases and offsets.  An offset whose spectrum is
 *   rho times the largest entry of that frequency keeps 22 bits while rho >= 2^-18; below that
 *   its own contribution carries a relative error of about 2^-40 / rho (1e-6 at rho = 1e-6,
 *   1e-5 at 1e-7; tests/test_gpu_parity.py::test_convolve_response_dynamic_range).  A response
 *   with a wider range between its offsets than that should use mac_mode 1 (fp32).
 *   Runs once per response and, unlike every other call, waits for the stream: the context
 *   has to know whether the response has the mirror symmetry R_{-i}^{-j} = R_i^j
 *   (exact equality is tested on the device).
 */
int tred_prepare_response(tred_ctx* ctx, const float* d_resp, float* d_rhat, void* stream);

/*
 * tred_convolve_plan -- footprints (O6).  Charge pixels: the (time slab, pixel)
 * pairs met by an occupied block; slab pixels: the (time slab, pixel) pairs met by the
 * output of an occupied block (charge pixels dilated by H); tiles: the (tile, pixel)
 * list the slab outputs overlap-add to.  All keys are (bt*npix_x + px)*npix_y + py, sorted.
 *   d_cp_keys   [cap_cp] int64 out, d_cp_off [NBt+1] int32 out (first index per slab), d_ncp
 *   d_sp_keys   [cap_sp] int64 out, d_sp_off [NBt+1] int32 out, d_nsp
 *   d_tile_keys [cap_tiles] int64 out, d_ntiles
 *   d_rt_off    [NBt+1] int32 out: first row tile of every slab (row tiles: runs of at most
 *               128 charge pixels of one slab and one 8-pixel-wide strip, the unit the
 *               tensor-core spectrum product works on; slot NBt = their number)
 *   d_plan_work at least tred_plan_work_bytes() bytes; its content (the index maps) is
 *               read again by tred_convolve and tred_gather_waveforms.
 */
size_t tred_plan_work_bytes(const tred_ctx* ctx);
int tred_convolve_plan(tred_ctx* ctx, int64_t nblocks, const int64_t* d_keys,
                       int64_t cap_cp, int64_t* d_cp_keys, int32_t* d_cp_off, int64_t* d_ncp,
                       int64_t cap_sp, int64_t* d_sp_keys, int32_t* d_sp_off, int64_t* d_nsp,
                       int64_t cap_tiles, int64_t* d_tile_keys, int64_t* d_ntiles,
                       int32_t* d_rt_off,
                       void* d_plan_work, size_t plan_work_bytes, void* stream);

/*
 * tred_convolve -- Eq. (12) evaluated as Eq. (14), pruned to
 * the time axis: real FFT along time of the S*S fine columns of every charge pixel
 * (zero where no block is occupied); per frequency, the product of the [charge pixels x
 * phases] spectra with the [phases x offsets] response spectrum (one batched complex
 * GEMM: tensor cores with split operands by default, fp32 FMA on request, see
 * tred_config.mac_mode); sum over the (2H+1)^2 offsets onto the output pixels in the
 * frequency domain (sum before the inverse FFT, Eq. (14)), in a fixed order -- in the default
 * mode inside the GEMM epilogue, per row tile, so the products never reach memory; one
 * inverse FFT per slab pixel.  Charge pixels are processed in chunks that fit the workspace;
 * results do not depend on the chunking (bit-identical).  No unordered float atomics.
 *   h_cp_off   [NBt+1] HOST copy of tred_convolve_plan's d_cp_off
 *   h_sp_off   [NBt+1] HOST copy of d_sp_off
 *   h_rt_off   [NBt+1] HOST copy of d_rt_off
 *   d_sp_data  [nsp][n_over*Bt] float32 out: current of (slab bt, pixel) from tick Bt*bt
 *   d_work     at least tred_convolve_work_bytes(min_rows) bytes with min_rows >= 1; more
 *              rows per chunk make larger launches.
 */
size_t tred_convolve_work_bytes(const tred_ctx* ctx, int64_t rows_chunk, int64_t nsp_batch);
int tred_convolve(tred_ctx* ctx, int64_t nblocks, const int64_t* d_keys, const float* d_payload,
                  const float* d_rhat,
                  int64_t ncp, const int64_t* d_cp_keys, const int32_t* h_cp_off,
                  int64_t nsp, const int64_t* d_sp_keys, const int32_t* h_sp_off,
                  const int32_t* h_rt_off,
                  const void* d_plan_work, float* d_sp_data,
                  void* d_work, size_t work_bytes, void* stream);

/*
 * tred_gather_waveforms -- overlap-add: every tile
 * (pixel, Tt = Bt ticks) is the sum, in ascending slab order, of the slab outputs that
 * cover it; optionally also writes dense rows for requested pixels.
 *   d_plan_work      plan of the blocks d_sp_data belongs to (its slab-pixel index map)
 *   d_tile_plan_work plan whose tile list d_tile_keys / d_tile_data follow (NULL: the same
 *                    plan).  A chunked run (config 4: bounded sets of occupied blocks,
 *                    PAPER.md:L242-250) makes one plan over all block keys for the tile
 *                    list and one per chunk of time slabs for the convolution.
 *   tile_begin, ntiles  the range of the tile list this call fills
 *   d_tile_keys [.] from tred_convolve_plan; d_tile_data [.][Bt] float32 in/out
 *   accumulate  0: tiles are overwritten; 1: the slab outputs are added onto the values
 *               already there (chunks processed in ascending slab order give the same
 *               sequence of additions, hence the same bits, as a single pass)
 *   d_pix_ids   [npix_req] int32 flat pixel ids px*npix_y+py (may be NULL if npix_req=0)
 *   d_dense     [npix_req][nticks] float32 out (may be NULL), read from d_tile_data
 */
int tred_gather_waveforms(tred_ctx* ctx, int64_t nsp, const float* d_sp_data,
                          const void* d_plan_work, const void* d_tile_plan_work,
                          int64_t tile_begin, int64_t ntiles, const int64_t* d_tile_keys,
                          float* d_tile_data, int accumulate,
                          int64_t npix_req, const int32_t* d_pix_ids, float* d_dense,
                          void* stream);

/*
 * tred_steps -- G4Step preprocessing (steps longer than a threshold, 5 mm in the
 * paper, are divided into step-segments that keep dE/dx; electrons that
 * survive recombination).  DESIGN.md readings G21 (n = ceil(len / max_len) equal pieces) and
 * G22 (the recombination law is the caller's choice; the paper gives none).  Needs no context.
 *   d_step   [8][nstep] float32 SoA rows x0,y0,z0,x1,y1,z1 (mm), dE (MeV), t0 (us)
 *   d_seg    [8][cap_seg] float32 out: the segment rows tred_drift reads (x0..z1, q electrons, t0),
 *            row stride cap_seg
 *   d_parent [cap_seg] int32 out: step every segment comes from
 *   d_nseg   int64 out: number of segments (may exceed cap_seg: TRED_ECAP semantics, nothing
 *            beyond the capacity is written)
 *   d_work   at least tred_steps_work_bytes(nstep) bytes
 * Piece counts come from fp64 round-to-nearest arithmetic in a fixed order (bit-exact).
 */
typedef struct tred_steps_config {
  double  max_len_mm;            /* threshold, PAPER.md:L57 (5 mm)                           */
  int32_t recomb_model;          /* 0 = Birks, 1 = modified box                              */
  double  w_ion_ev;              /* energy per electron-ion pair (eV)                        */
  double  efield_kv_cm, density_g_cm3;
  double  birks_A, birks_k;      /* R = A / (1 + k/(rho E) dE/dx)                            */
  double  box_alpha, box_beta;   /* R = ln(alpha + b dE/dx)/(b dE/dx), b = beta/(rho E)      */
} tred_steps_config;

size_t tred_steps_work_bytes(int64_t nstep);
int tred_steps(const tred_steps_config* cfg, int64_t nstep, const float* d_step, int64_t cap_seg,
               float* d_seg, int32_t* d_parent, int64_t* d_nseg, void* d_work, size_t work_bytes,
               void* stream);

/*
 * tred_steps_static -- tred_steps without a workspace argument and without any allocation: the
 * same operation (readings G21, G22), the same arithmetic in the same order,
 * the same bits in d_seg / d_parent / d_nseg, for callers that cannot provide d_work.
 *
 * Who needs it.  The step splitter sits in front of the simulation, typically in an input stage
 * that owns no device workspace and cannot get one from the CUDA runtime: all device memory of
 * the job was given to a pool at start-up; or another thread of the process is recording a CUDA
 * graph in the default capture mode, during which cudaMalloc / cudaFree from ANY thread are
 * errors that also ruin that recording; or the caller is a per-event loop that cannot take the
 * device-wide synchronisation cudaMalloc / cudaFree imply.  The call and everything under it
 * make no cudaMalloc, cudaFree or other allocating call, on the first call or later.
 *
 * How.  Its scratch (first segment of every step + the block sums of the scan) is a fixed
 * __device__ array inside libtred.so, TRED_STEPS_STATIC_BYTES long.  Consequences to know:
 *   - limit: nstep <= TRED_STEPS_STATIC_MAX (= tred_steps_static_max()).  More returns TRED_ECAP
 *     before anything is enqueued and leaves the outputs untouched: split the batch (segments of
 *     different steps are independent; add the batch's first step index to d_parent), or use
 *     tred_steps with a workspace;
 *   - cost: every GPU on which the process has loaded libtred.so holds those ~4 MiB until the
 *     process ends, whether or not this call is ever made;
 *   - sharing: all calls on one device use the one array.  Calls on the same stream follow each
 *     other and are fine (nothing needs clearing between them: a call writes every scratch entry
 *     it later reads).  Calls that may run on the GPU at the same time -- different streams, or
 *     several host threads with their own streams -- overwrite each other's scratch and give
 *     wrong results: order them with events or keep one stream for this call per device;
 *   - first call on a device: looks up the array's address on that device (cudaGetSymbolAddress,
 *     with the device current; kept per device afterwards, under a mutex).  Make that first call
 *     during set-up, before any stream capture is begun anywhere in the process.
 * Arguments as for tred_steps, minus d_work / work_bytes; cap_seg = 0 is the counting pass.
 */
#define TRED_STEPS_STATIC_MAX   1048576      /* steps per call                                  */
#define TRED_STEPS_STATIC_BYTES 4196608      /* (MAX + 1) int32 rounded to 256, + 2048 for the scan */
int64_t tred_steps_static_max(void);
int tred_steps_static(const tred_steps_config* cfg, int64_t nstep, const float* d_step, int64_t cap_seg,
                      float* d_seg, int32_t* d_parent, int64_t* d_nseg, void* stream);

/*
 * tred_readout -- trigger-reset pixel readout (Fig. 4; noise terms
 * PAPER.md:L262; reading G23).  Per channel, tick by tick: the charge on the
 * preamplifier is the running fp32 sum of the current; when it reaches threshold_e (+ the
 * discriminator noise draw of this hit) the channel integrates n_integ more ticks and records
 * (tick of digitisation, charge + preamplifier noise draw); it is then reset to the baseline
 * draw and dead for n_reset ticks.  A hit whose digitisation tick falls outside the window
 * is lost; at most max_hits records per channel.
 *   d_wave     [npix][nticks] float32 current in electrons per tick (rows of d_dense of
 *              tred_gather_waveforms)
 *   d_noise    [npix][max_hits][3] float32 draws (discriminator, preamplifier, baseline) in
 *              electrons for every possible hit, or NULL for none: random numbers are inputs
 *   d_nhit     [npix] int32 out; d_hit_tick [npix][max_hits] int32 out (-1 = unused);
 *   d_hit_adc  [npix][max_hits] float32 out (rounded to adc_lsb_e electrons if > 0)
 */
typedef struct tred_readout_config {
  double  threshold_e;           /* discriminator threshold, electrons                      */
  int32_t n_integ;               /* fixed integration after the crossing, ticks             */
  int32_t n_reset;               /* dead ticks after the digitisation                        */
  int32_t max_hits;              /* capacity of the per-channel record list                 */
  double  adc_lsb_e;             /* 0: keep the charge as it is; > 0: round to this step     */
} tred_readout_config;

int tred_readout(const tred_readout_config* cfg, int64_t npix, int32_t nticks, const float* d_wave,
                 const float* d_noise, int32_t* d_nhit, int32_t* d_hit_tick, float* d_hit_adc,
                 void* stream);

/*
 * tred_simulate -- the whole path in one call: segments in, per-pixel current waveforms out
 * (Fig. 1): tred_drift, tred_blockbin, tred_convolve_plan, tred_effq,
 * tred_convolve, tred_gather_waveforms on buffers carved from one caller-provided workspace.
 *   seg          [8][nseg] float32 as for tred_drift, in HOST memory if seg_on_host != 0 (copied
 *                to the device by the call), else in device memory
 *   d_rhat       from tred_prepare_response
 *   payload_budget_bytes  0: the block payload of the whole event is held at once.  > 0 and smaller
 *                than the payload: the event is processed in ranges of time slabs whose payload
 *                fits (chunks bounded by device memory; BASELINE config 4); the
 *                result is bit-identical to one pass (a slab's output depends on that slab's
 *                blocks only, and the overlap-add continues the running sum in slab order)
 *   d_work       device workspace, work_bytes long.  Too small: TRED_ECAP with
 *                h_result->work_bytes_needed set.  Once the counts of the event have been read
 *                (h_result->nblocks > 0) that number is enough for this event in the unchunked
 *                form; a workspace too small even for the lists that precede the read (drift
 *                records, pair lists, plan: h_result->nblocks == 0), and every TRED_ECAP of the
 *                chunked form, report what is known at that point plus a margin (64 MiB / 6 GiB),
 *                so a caller that grows the workspace by the reported size may see TRED_ECAP up
 *                to three times for one event.  h_result is zeroed first on every return
 *   tile_keys    [cap_tiles] int64 out, tile_data [cap_tiles][Bt] float32 out: the waveform tiles,
 *                keys ascending, in HOST memory if out_on_host != 0, else device memory.
 *                h_result->ntiles > cap_tiles: TRED_ECAP, nothing written
 *   d_pix_ids, d_dense  optional dense rows as for tred_gather_waveforms (device memory)
 *   h_result     HOST, filled by the call
 * Host waits: the call reads the device-side counts ONCE per event (pairs, blocks, footprints
 * and per-slab offsets in one copy, after the plan), plus once per slab range in the chunked
 * form.  The capacities of the lists that precede that read come from the previous event on
 * this context (first event, or an event that outgrows them: one more read).  The outputs are
 * complete when `stream` has finished.
 */
typedef struct tred_sim_result {
  int64_t nseg, npairs, nblocks, ncp, nsp, ntiles, nrt, nchunks;
  int64_t work_bytes_needed;     /* set with TRED_ECAP when d_work is too small           */
  int64_t conv_bytes_needed;     /* of which: what tred_convolve would like (it chunks the charge
                                    pixels to what it gets) and the least it can work with; a
                                    caller bounding peak memory may grant anything in between  */
  int64_t conv_bytes_min;
  int64_t work_bytes_used;
  int32_t host_reads;            /* device-to-host reads of counts this call made           */
  int32_t mac_mode;              /* tred_last_mac_mode                                      */
} tred_sim_result;

int tred_simulate(tred_ctx* ctx, int64_t nseg, const float* seg, int seg_on_host, const float* d_rhat,
                  int64_t payload_budget_bytes, void* d_work, size_t work_bytes,
                  int64_t cap_tiles, int64_t* tile_keys, float* tile_data, int out_on_host,
                  int64_t npix_req, const int32_t* d_pix_ids, float* d_dense,
                  tred_sim_result* h_result, void* stream);

/*
 * tred_truth -- truth record ("segment-id -> charge per (channel, short time
 * slice)"; reading G24): the effective charge of every segment summed over the grid
 * points of each pixel and each time tile (Bt ticks) of its clipped footprint.  One entry per
 * (pixel, tile) the footprint reaches, ordered by segment, then by key.
 *   d_augf, d_augi  from tred_drift
 *   d_rec_seg [cap_rec] int32 out, d_rec_key [cap_rec] int64 out ((tile * npix_x + px) * npix_y + py,
 *             the key of tred_convolve_plan's tiles), d_rec_q [cap_rec] float32 out (electrons)
 *   d_nrec    int64 out: number of entries (TRED_ECAP semantics: may exceed cap_rec, nothing
 *             beyond the capacity is written)
 *   d_work    at least tred_truth_work_bytes(nseg) bytes
 * A record holds at most 32 pixels and 32 time tiles per axis (a segment of the paper's
 * workloads reaches 2-4).  If any segment reaches more, *d_nrec is set to -1 and the entries
 * written are not to be used: nothing is truncated silently.
 */
size_t tred_truth_work_bytes(const tred_ctx* ctx, int64_t nseg);
int tred_truth(tred_ctx* ctx, int64_t nseg, const float* d_augf, const int32_t* d_augi, int64_t cap_rec,
               int32_t* d_rec_seg, int64_t* d_rec_key, float* d_rec_q, int64_t* d_nrec, void* d_work,
               size_t work_bytes, void* stream);

/*
 * Stage profiling (the paper's "profiler-guided optimization", Fig. 10).
 * tred_profile_begin clears the counters; with record_events != 0 every stage of the
 * following calls is bracketed by CUDA events on the launching stream.
 * tred_profile_end synchronises those events (the one place the library waits on the
 * device, on request) and returns, per stage, the summed milliseconds (0 if events were
 * off) and the number of kernels launched.  Stage s is named tred_stage_name(s),
 * s < tred_stage_count().  h_ms / h_launches: HOST arrays of nstage entries.
 */
int tred_profile_begin(tred_ctx* ctx, int record_events);
/* Measurement aid, not part of the path: enqueues one kernel of nothing but independent fp32
 * FMA chains (8 per thread, 64 x iters FMAs each, 8 CTAs of 256 threads per SM) and writes the
 * floating-point operations it executes to *h_flops (host).  Timed by the caller (CUDA events
 * on `stream`) it gives the fp32 FMA rate this device sustains, the peak of the "alu"
 * rooflines.  d_out: at least one float of device memory. */
int tred_bench_fma(tred_ctx* ctx, int32_t iters, float* d_out, double* h_flops, void* stream);
int tred_profile_end(tred_ctx* ctx, int nstage, float* h_ms, int64_t* h_launches);
int tred_stage_count(void);
const char* tred_stage_name(int stage);

#ifdef __cplusplus
}
#endif
#endif /* TRED_H */
