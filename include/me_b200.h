/* me_b200.h -- C ABI of the B200 matrix-element library (libme_b200.so).
 *
 * The boundary follows the paper's statement of the problem: a "multi-event API" made of "reentrant
 * stateless functions with well-defined input and output data" (Fig. 1 caption)
 * that can be used "as a CUDACPP ME library ... in frameworks other than MG5aMC":
 * momenta[nevt][npar][4] (fp64) plus the per-event strong coupling in, ME[nevt] out, plus optional
 * per-event helicity and colour selection from supplied uniform random numbers (BASELINE.json
 * north_star).  What is computed: "from the particle momenta, the matrix element (ME) ... is computed"
 * as Feynman diagrams + the colour-matrix quadratic form, summed over
 * helicity combinations:
 *
 *     ME = (1/denom) * sum_{h good} sum_{s,t} conj(J_s(h)) C_st J_t(h)
 *
 * Conventions (readings R1-R16)
 *   - all `d_*` arguments are DEVICE pointers owned by the caller (8-byte aligned; int32 outputs 4-byte);
 *     everything else is a HOST pointer.  `stream` is a cudaStream_t passed as void*; work is enqueued
 *     on it and NOT synchronised unless stated.  Device memory the library allocates: a 1 KB table in me_create;
 *     the selection scratch of the small processes in me_filter_helicities / me_set_good_helicities; staging in
 *     me_compute_host (grows only); and, for gg_ttgg / gg_ttggg, the pipeline scratch that holds a chunk of events
 *     between the three kernels of the path (23 KB per gg_ttgg event, 245 KB per gg_ttggg event in fp64).  That
 *     scratch follows the batch size: me_reserve sizes it up front; otherwise me_filter_helicities / me_compute grow
 *     it (cudaFree + cudaMalloc, which waits for the device) when a batch LARGER than any before arrives, up to 2 GiB (gg_ttgg) or
 *     8 GiB (gg_ttggg) per handle, beyond which a batch runs in more chunks.  A call no larger than an earlier one, or than what me_reserve
 *     was given, never allocates.  me_destroy frees everything.  Every call makes
 *     the handle's device current while it runs and restores the caller's current device before returning.
 *   - one handle serves one stream at a time: calls on the same handle from different streams must not overlap
 *     on the device (the scratch is per handle); use one handle per stream for concurrency.
 *   - momenta: [nevt][npar][4] doubles, (E, px, py, pz) in GeV, particle order = process string order,
 *     particles 0,1 incoming; for the gg processes 2 = t, 3 = tbar, 4.. = g; for gux_taptamggux
 *     (g ubar -> tau+ tau- g g ubar through a photon or a Z, the mixed EW+QCD class of PAPER.md:110-122 Table 4)
 *     0 = g, 1 = ubar, 2 = tau+, 3 = tau-, 4,5 = g, 6 = ubar; for ee_mumu
 *     0 = e+, 1 = e-, 2 = mu+, 3 = mu-.  No special frame is assumed.
 *   - gs: [nevt] doubles, g_s = sqrt(4 pi alpha_s) per event (ignored by ee_mumu, may be NULL there).
 *   - helicity index h (0-based): row of the table returned by me_helicity_table; row h has
 *     lambda_k = +1 if bit (npar-1-k) of h is set, else -1 (particle 0 slowest).
 *   - colour index c (0-based): row of me_color_table, the permutations of the gluon particle indices
 *     in lexicographic order (string from t to tbar; gux_taptamggux: from the incoming to the outgoing ubar).
 *     ee_mumu: ncol = 1.
 *   - every function returns 0 on success or a negative ME_ERR_* code; me_last_error gives a
 *     NUL-terminated description of the last failure of that handle (or of me_create if h == NULL).
 *     No C++ exception crosses the boundary.  A handle may be used from one host thread at a time;
 *     different handles are independent.
 */
#ifndef ME_B200_H
#define ME_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct me_handle me_handle;

/* physics parameters; NULL in me_create selects the BASELINE.json values */
typedef struct me_params {
  double mt;    /* top mass [GeV]                      173.0     */
  double wt;    /* top width [GeV], fixed-width scheme 1.4915    */
  double mz;    /* Z mass [GeV]                        91.188    */
  double wz;    /* Z width [GeV]                       2.441     */
  double aewm1; /* 1/alpha_EM                          132.507   */
  double gf;    /* Fermi constant [GeV^-2]             1.16639e-5 */
} me_params;

enum { ME_FP64 = 0, ME_FP32 = 1, ME_MIXED = 2 };

enum {
  ME_OK = 0,
  ME_ERR_ARG = -1,        /* NULL / misaligned pointer, negative nevt, bad enum */
  ME_ERR_PROCESS = -2,    /* unknown process name */
  ME_ERR_NO_HELICITIES = -3, /* me_compute before me_filter_helicities / me_set_good_helicities */
  ME_ERR_CUDA = -4,       /* CUDA runtime error (text in me_last_error) */
  ME_ERR_NOMEM = -5
};

/* process: "ee_mumu" | "gg_tt" | "gg_ttg" | "gg_ttgg" | "gg_ttggg" | "gux_taptamux" | "gux_taptamgux" | "gux_taptamggux"
 * (g ubar -> tau+ tau- ubar + 0, 1, 2 further gluons); precision: ME_FP64/ME_FP32/ME_MIXED
 * (mixed = Feynman diagrams in fp64, colour quadratic form in fp32); device: CUDA ordinal. */
int me_create(me_handle** out, const char* process, int precision, const me_params* params, int device);
int me_destroy(me_handle* h);
const char* me_last_error(const me_handle* h);

/* sizes: any output pointer may be NULL */
int me_info(const me_handle* h, int* npar, int* ncomb, int* ncol, int* ndiag, int* denom);
/* out[ncomb][npar], entries +-1 */
int me_helicity_table(const me_handle* h, int8_t* out);
/* out[ncol][ngluon]: gluon particle indices in string order (nothing written for ee_mumu) */
int me_color_table(const me_handle* h, int8_t* out);
/* out[ncol][ncol], the real symmetric colour matrix C */
int me_color_matrix(const me_handle* h, double* out);

/* One-time good-helicity filter (BASELINE.json north_star (e); reading R10): evaluates ALL helicities in
 * fp64 on the first min(nevt, 16384) events and keeps h iff max_e |M_h|^2 / sum_h' |M_h'|^2 > 1e-12.
 * Synchronises the stream (it is an initialisation call). */
int me_filter_helicities(me_handle* h, const double* d_momenta, const double* d_gs, int64_t nevt, void* stream);
/* mask[ncomb], 1 = good */
int me_get_good_helicities(const me_handle* h, int* ngood, uint8_t* mask);
int me_set_good_helicities(me_handle* h, const uint8_t* mask);

/* Sizes the pipeline scratch of a gg_ttgg / gg_ttggg handle for calls of up to max_events_per_call events (at most
 * 2 GiB / 8 GiB; see the conventions above), so that no later me_filter_helicities / me_compute of that size allocates.  Costs
 * nothing for the other processes.  May be called before or after the helicity filter; never shrinks. */
int me_reserve(me_handle* h, int64_t max_events_per_call);

/* The hot path.  d_me[nevt] receives ME (fp64 in every build).  If d_rndhel and d_selhel are given,
 * d_selhel[nevt] receives the first good h with r_hel * S < sum_{h' <= h} |M_h'|^2 (last good one if
 * rounding leaves none); likewise d_rndcol/d_selcol with the weights w_c = sum_{h good} |J_c(h)|^2
 * (reading R11).  Enqueues on `stream`, does not synchronise, allocates nothing in steady state (see me_reserve). */
int me_compute(me_handle* h, const double* d_momenta, const double* d_gs, const double* d_rndhel,
               const double* d_rndcol, int64_t nevt, double* d_me, int32_t* d_selhel, int32_t* d_selcol,
               void* stream);

/* The hot path for callers that must not allocate device memory: gg -> t tbar g (the process "gg_ttg", particle order
 * g g -> t tbar g), fp64, with the same optional helicity / colour selection and the same arithmetic as me_compute.
 *
 * Why it exists.  me_create and me_set_good_helicities call cudaMalloc.  Some callers cannot: a host application
 * that has given the whole GPU to its own memory pool at start-up (a library's cudaMalloc then fails, or breaks the
 * application's accounting), a process confined to a fixed device-memory budget, or a loop that shares the GPU with
 * other streams and cannot afford the device-wide stall an allocation may cause.  This function takes no handle and
 * calls no cudaMalloc, cudaFree or allocating library routine, ever.  The scratch its kernel needs (the running sums
 * over the good helicities, one double per helicity and event) is a fixed 4 MiB array inside the library's device
 * image; every GPU that loads libme_b200.so holds those 4 MiB until the process exits, used or not.  (Register-spill
 * space of the kernel, 1.7 KB per thread, is the CUDA driver's own business at the first launch, as for any kernel.)
 *
 * Limit.  nevt <= ME_NOALLOC_MAX_EVENTS (16384, the paper's typical 8k-16k events per launch); a larger
 * nevt is refused with ME_ERR_ARG and a message saying so -- split the batch into calls on the same stream.
 *
 * Arguments.  params: as in me_create (NULL = defaults; only mt and wt matter).  good_mask: [32] bytes, 1 = helicity
 * combination kept (me_get_good_helicities of any gg_ttg handle, in any process, gives it; for a massive top all 32
 * pass), NULL = all 32.  The d_* pointers, nevt and stream: as in me_compute; d_gs is required.  errbuf / errcap:
 * HOST buffer that receives a NUL-terminated message on failure (may be NULL; there is no handle to ask).
 * Returns 0 or a negative ME_ERR_* code.  Enqueues one kernel on `stream`, does not synchronise.
 *
 * Device.  Works on the device that is current in the calling thread; the buffers and the stream must belong to it.
 * The first call on each device looks up the device address of the static scratch (cudaGetSymbolAddress, no
 * allocation); make that first call before any stream capture begins.
 *
 * Sharing.  All calls on a device use the same scratch array, and it keeps whatever the last call left there.  Nothing
 * in it needs clearing: every thread writes its own entries before reading them.  But two calls of one process whose
 * kernels run at the same time on one GPU (issued on different streams, from one host thread or several) overwrite
 * each other's sums and return wrong selections: issue the calls of one device on one stream, or order them with
 * events.  d_me is not affected, only d_selhel.  Different processes each have their own copy of the array. */
#define ME_NOALLOC_MAX_EVENTS 16384
int me_compute_noalloc(const me_params* params, const uint8_t* good_mask, const double* d_momenta, const double* d_gs,
                       const double* d_rndhel, const double* d_rndcol, int64_t nevt, double* d_me, int32_t* d_selhel,
                       int32_t* d_selcol, void* stream, char* errbuf, int errcap);

/* Multichannel running ("events from different channels" in one launch).  Reading
 * R17 of DESIGN.md (the paper gives no formula): a channel is a Feynman diagram of the process; channels are numbered
 * 0 .. ndiag-1 in increasing byte order of the structural keys returned by me_channel_table.  d_channel[nevt] (device,
 * int32, values outside 0 .. ndiag-1 are clamped for the colour selection and give num = 0) assigns a channel to every
 * event; events of any mix of channels may share a call (a warp never works on two events at once in the kernels that
 * look at the channel).  Outputs, beside those of me_compute:
 *   d_num[nevt] = sum over the good helicities and the colour-structure terms of diagram d = channel[e] of |A_d|^2,
 *   d_den[nevt] = the same summed over ALL diagrams   (fp64 in every build; both include g_s^(2n)),
 * so that num/den is the single-diagram-enhancement weight of the event's channel; and the colour selection
 * (d_selcol) only picks flows that diagram d contributes to.  d_me is the plain ME (multiply by num/den yourself).
 * gg processes only (ME_ERR_PROCESS for ee_mumu and gux_taptamggux).  The first call allocates the kernel's per-event scratch
 * (3.6 KB x min(nevt, 65536) at most); later calls with no more events do not allocate.  Enqueues on `stream`. */
int me_compute_multichannel(me_handle* h, const double* d_momenta, const double* d_gs, const double* d_rndhel,
                            const double* d_rndcol, const int32_t* d_channel, int64_t nevt, double* d_me,
                            int32_t* d_selhel, int32_t* d_selcol, double* d_num, double* d_den, void* stream);
/* Channel keys, one per line in channel order, NUL terminated: the trees attached to the quark line from t to tbar
 * separated by "|"; a leaf is its particle index, "(A,B)" a three-gluon vertex, "[A,B,C]" a four-gluon vertex.
 * Returns the bytes needed (call with out = NULL first), or a negative error code. */
int me_channel_table(const me_handle* h, char* out, int cap);

/* Same call with HOST buffers (pinned or pageable): copies in, computes, copies out and synchronises.  The batch
 * flows in chunks through two device staging slots on three internal streams, so that the copies of neighbouring
 * chunks overlap the kernels (pinned host memory needed for that; pageable memory still works, serially).
 * This is the end-to-end path bench.py times as `e2e`. */
int me_compute_host(me_handle* h, const double* momenta, const double* gs, const double* rndhel,
                    const double* rndcol, int64_t nevt, double* me, int32_t* selhel, int32_t* selcol);

/* Device-side seeded inputs (the paper's standalone application draws random numbers and
 * maps them to momenta with a phase-space sampling algorithm).  Writes, for the events
 * start .. start+nevt-1 of the seeded stream, d_momenta[nevt][npar][4] (incoming p0 = (E,0,0,E), p1 = (E,0,0,-E),
 * E = sqrts/2; final state from RAMBO flat phase space with the process' masses) and, where the pointer is not
 * NULL, d_gs[nevt] (alphas > 0: g_s = sqrt(4 pi alphas) fixed; alphas <= 0: alpha_s ~ U[0.10, 0.13] per event),
 * d_rndhel[nevt], d_rndcol[nevt] (uniforms in (0,1)) and d_weight[nevt] (the RAMBO phase-space weight).  The
 * generator is counter-based (splitmix64 steps on (seed, stream, event index): event e of a stream is the same
 * whatever the batch it is made in); its numpy oracle is oracle/rambo.py (tests/test_gpu_rambo.py).  Enqueues on `stream`, does not synchronise. */
int me_generate(me_handle* h, uint64_t seed, int64_t start, int64_t nevt, double sqrts, double alphas,
                double* d_momenta, double* d_gs, double* d_rndhel, double* d_rndcol, double* d_weight, void* stream);

/* launch geometry of the last me_compute (for reports): threads per block, blocks, registers per thread,
 * bytes of local (spill) memory per thread of the dominant kernel (gg_ttgg / gg_ttggg: the amplitude kernel) */
int me_launch_info(const me_handle* h, int* threads, int* blocks, int* regs, int* local_bytes);

/* Kernels enqueued by the last me_compute (3 per chunk for gg_ttgg / gg_ttggg: setup, amplitudes, colour contraction;
 * 1 otherwise), the events per chunk and the bytes of pipeline scratch the handle owns (0 if it has none) */
int me_launch_stats(const me_handle* h, int* launches, int64_t* chunk_events, int64_t* scratch_bytes);

/* Measured FMA peak of the device: a register-resident dependent-FMA-chain microbenchmark (best of 5
 * launches of a few ms, synchronous).  precision ME_FP64 or ME_FP32; *tflops receives TFLOP/s with
 * FMA = 2 FLOP.  This is the denominator of the roofline fractions. */
int me_fma_peak(int precision, int device, double* tflops);

/* Measured peak of the tensor-core instructions the colour contraction uses (same kind of microbenchmark):
 * kind 0 = mma.sync m8n8k4 f64 (DMMA: on B200 it runs on the FP64 units, so it buys no throughput over DFMA, only
 * issue slots), kind 1 = mma.sync m16n8k8 tf32 with fp32 accumulation (a pipe of its own).  *tflops: 2 m n k FLOP
 * per warp-wide MMA.  Context for the roofline of bench.py (north_star (d): tensor cores "only where it
 * genuinely batches"). */
int me_mma_peak(int kind, int device, double* tflops);

#ifdef __cplusplus
}
#endif
#endif
