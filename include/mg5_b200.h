/* mg5_b200.h -- C ABI of the B200-native leading-order matrix-element engine.
 *
 * What the library computes (arxiv 2510.05392; citations are /root/reference/PAPER.md lines):
 *   "takes as input an array of particle momenta for many events (i.e. 4*npar fptype values for each of
 *    nevt events), and returns as its output an array of matrix elements (i.e. one fptype value for each
 *    of nevt events)"                                                        (Sec. 2.2)
 *   me[e] = (1/denom) sum_{good helicities h} Re( J_h(e)^dagger C J_h(e) )   (PAPER.md:95-98, 117-119, 124,
 *    Eq. 1 at PAPER.md:264-269), J_h(e) = the ncolor dual amplitudes ("jamps") summed over the process's
 *    Feynman diagrams.
 *
 * Conventions
 *   - All functions return MG_OK (0) or a negative MG_E* code; nothing throws across this boundary.
 *     mg_last_error() gives a text for the last failure on that handle (or for a failed init when NULL).
 *   - Pointers are marked HOST or DEVICE.  The caller owns every buffer it passes; the library owns only
 *     the opaque handle, its constant tables, and its internal CUDA streams/events.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Calls that take a
 *     stream are asynchronous and stream-ordered unless stated otherwise.
 *   - Momenta: fp64, array-of-structures momenta[nevt][npar][4] = (E, px, py, pz) in GeV; particle order =
 *     order in the process string (two beams along +z/-z, then the final state); all physical (E > 0).
 *   - Helicity index h = sum_i b_i 2^(npar-1-i), b_i = 0 <-> helicity -1, 1 <-> +1, particle 0 most
 *     significant (reading A2).
 *   - Device must be compute capability 10.x (B200, sm_100a): MG_ENODEV otherwise.  There is no CPU path.
 */
#ifndef MG5_B200_H
#define MG5_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mg_process mg_process; /* opaque, library-owned */

/* the paper's FPTYPE d / m / f: amplitudes fp64 + colour sum fp64; amplitudes fp64 +
 * colour sum fp32/TF32; everything fp32 */
enum { MG_FP64 = 0, MG_MIXED = 1, MG_FP32 = 2 };
enum { MG_OK = 0, MG_EINVAL = -1, MG_ENODEV = -2, MG_ENOMEM = -3, MG_ECUDA = -4, MG_ESTATE = -5 };

/* colour-sum implementations ("color_sum_kernel" vs "color_sum_blas", here own kernels):
 *   MG_CS_FUSED  : inside the diagram kernel, scalar ALUs, triangular form; jamps never leave the thread
 *   MG_CS_TENSOR : jamps written to the workspace as [2][ncolor][nGoodHel*nevt], then ONE
 *                  tensor-core contraction over all helicities: DMMA (mma.sync f64) in MG_FP64,
 *                  tcgen05 kind::tf32 with TMEM accumulators in MG_MIXED / MG_FP32 */
enum { MG_CS_FUSED = 0, MG_CS_TENSOR = 1 };

/* helicity scheduling ("helicity streams"):
 *   MG_SCHED_GRID    : helicity is a grid dimension of one launch (default)
 *   MG_SCHED_STREAMS : one launch per good helicity, each on its own library-owned stream, forked from and
 *                      joined back into the caller's stream with events */
enum { MG_SCHED_GRID = 0, MG_SCHED_STREAMS = 1 };

/* diagram stage:
 *   MG_DIAG_THREAD : one thread per (event, helicity), the paper's layout
 *   MG_DIAG_SHARED : one CTA per event, all helicities at once; wavefunctions shared between helicities in shared
 *                    memory, jamps written to the workspace and contracted by the colour-sum kernel (g g -> t tbar +
 *                    2 or 3 gluons, MG_FP64 / MG_MIXED; the default there; g g -> t tbar + 4 gluons: the only kernel) */
enum { MG_DIAG_THREAD = 0, MG_DIAG_SHARED = 1 };

/* Create a process.  name: "epem_mupmum", "gg_ttx", "gg_ttxg", "gg_ttxgg", "gg_ttxggg" (BASELINE.json configs;
 * Table 2), or "gg_ttxgggg" (g g -> t tbar g g g g, Table 2's 2 -> 6 row: 15 495 diagrams, 720 colour
 * flows, 256 helicities; Tables 5-8).  The latter runs with MG_DIAG_SHARED only (generic
 * helicity-shared kernel, the event's wavefunctions in a per-CTA scratch area in global memory owned by the handle: about
 * 0.5 GB of device memory per handle) in MG_FP64 (720-colour FP64 tensor-core colour sum) and MG_MIXED (the same on tcgen05
 * kind::tf32); MG_FP32 -> MG_EINVAL.
 * Parameters start at the BASELINE.json card.  *out is NULL on failure. */
int mg_init_process(const char* name, int precision, int device, mg_process** out);

/* Static facts about the process (any pointer may be NULL). ngroups = diagram-group functions in the diagram
 * kernel. */
int mg_process_info(const mg_process* p, int* npar, int* ncomb, int* ncolor, int* ndiagrams, int* ngroups);

/* Algorithmic floating-point operations of the diagram stage per (event, helicity) and of the colour sum per
 * (event, helicity) (dense 2*2*ncolor^2 + 4*ncolor), as counted by the generator. */
int mg_process_flops(const mg_process* p, double* diagram_flops, double* color_flops);

/* Set model parameters.  keys (HOST strings): "aEWM1" (1/alpha), "mZ", "wZ", "mW", "mT", "wT", "aS".
 * Derived couplings are recomputed on the host.  Unknown key -> MG_EINVAL, nothing changed. */
int mg_set_parameters(mg_process* p, const char* const* keys, const double* values, int n);

/* Options: "color_sum" (MG_CS_*), "schedule" (MG_SCHED_*), "diagrams" (MG_DIAG_*), "block" (threads per block of the
 * MG_DIAG_THREAD kernel, multiple of 32, <= 256; default 64, the fastest of 32..256 on B200 for g g -> t tbar (g)),
 * "hs_color_alu" (MG_DIAG_SHARED in MG_MIXED: 1 = scalar-ALU fp32 colour-sum kernel instead of the tcgen05 one),
 * "tf32_direct" (MG_DIAG_SHARED in MG_MIXED with the tcgen05 kernel, default 1: the diagram kernel writes the jamps as TF32
 * values straight in the tensor-core operand layout and the contraction accumulates J Lhi + J Llo; 0: fp32 jamps, two-term
 * split of J inside the contraction, three products),
 * "jamp_chunk_mib" (size of the jamps buffer inside the workspace; default 16384 = every BASELINE.json batch in one chunk;
 * smaller values trade workspace for more launches), "timing" (0/1),
 * "max_streams" (MG_SCHED_STREAMS: helicities share this many streams round robin, 0 = one each),
 * "graph" (1: the launch sequence of a batch is captured into a CUDA graph on its first execution and replayed while the
 * arguments and the handle's state are unchanged; ignored while "timing" = 1; mg_get_option
 * "graph_replays" counts the replays of the current graph; mg_get_option "probe_events" = the number of events of the first
 * batch the automatic helicity filter looks at, at most: 1024, or 16 for "gg_ttxgggg" whose probe goes through the jamps buffer),
 * "p3_tensor" ("gg_ttxgggg" only, default 1: the generic kernel contracts the pair objects with the largest branch -- phase 3,
 * the sum over the entries of a colour flow for all 256 helicity combinations -- on the FP64 tensor path, mma.sync.m8n8k4.f64;
 * 0: on the FP64 ALU, thread = helicity combination; same numbers up to the order of the sum; MG_EINVAL for other processes).
 * With "diagrams" = MG_DIAG_SHARED the jamps always go through the workspace and the tensor-core colour sum ("color_sum" and
 * "block" then only affect the helicity filter and MG_DIAG_THREAD).
 * Unknown key, bad value, or a combination that cannot run (helicity streams with the MG_DIAG_SHARED kernel, which has
 * no per-helicity launches) -> MG_EINVAL, nothing changed. */
int mg_set_option(mg_process* p, const char* key, int value);
/* Current value of an option (same keys).  Unknown key -> MG_EINVAL. */
int mg_get_option(const mg_process* p, const char* key, int* value);

/* Bytes of DEVICE workspace needed by mg_sigma_batch / mg_helicity_filter for batches of up to nevt events
 * with the current options and good-helicity list (all ncomb helicities if none is set yet).
 * Layout inside is private; 256-byte alignment of the base is required. */
size_t mg_workspace_bytes(const mg_process* p, int nevt);

/* Helicity filter ("a pre-determined set of good helicities whose contribution is non-zero",
 * PAPER.md:649).  Evaluates every helicity combination on the first nprobe events of d_momenta (DEVICE),
 * all in one launch, and marks h good iff max_e me_h(e)/sum_h' me_h'(e) > 1e-8 (reading A5).
 * h_mask (HOST, [ncomb], out) and ngood (HOST, out) may be NULL.  Synchronises the stream.  The list is
 * stored in the handle. */
int mg_helicity_filter(mg_process* p, const double* d_momenta, int nprobe, void* d_workspace, size_t ws_bytes,
                       void* cuda_stream, unsigned char* h_mask, int* ngood);

/* Install a good-helicity mask directly (HOST, [ncomb]); all ones = the paper's
 * CUDACPP_RUNTIME_GOODHELICITIES=ALL. */
int mg_set_good_helicities(mg_process* p, const unsigned char* h_mask);

/* One batch: d_momenta (DEVICE, [nevt][npar][4] fp64) -> d_me (DEVICE, [nevt] fp64, GeV^(-2(npar-4))).
 * If no good-helicity list is set, the filter runs first on min(nevt, 1024) events (this synchronises).
 * ws_bytes must be >= mg_workspace_bytes(p, nevt).  nevt = 0 is a no-op. */
int mg_sigma_batch(mg_process* p, const double* d_momenta, int nevt, double* d_me, void* d_workspace,
                   size_t ws_bytes, void* cuda_stream);

/* The rest of the paper's ME-engine interface (the engine "also receives other inputs": an event-by-event
 * running alpha_s(Q^2), and "two random numbers for each event", from which it selects "a color and a helicity for event
 * ievt" -- Table 1; the alpha_s-dependent couplings are computed in a kernel of their own).
 * All extra pointers are DEVICE arrays of nevt elements and may be NULL (then this is mg_sigma_batch):
 *   d_alphas : alpha_s of each event.  The couplings kernel computes G = sqrt(4 pi alpha_s(e)); every diagram of the g g ->
 *              t tbar + gluons processes carries G^n, so d_me[e] is the card's matrix element times (alpha_s(e)/aS)^n
 *              (e+ e- -> mu+ mu- does not depend on it).
 *   d_rndhel, d_selhel : uniform numbers in [0, 1) -> helicity index h (numbering above) of the first good helicity k, in
 *              increasing h, with  rnd * sum_j me_hj < sum_{j <= k} me_hj  (reading A15).
 *   d_rndcol, d_selcol : -> colour flow c (index of the permutation sigma in lexicographic order, the order of
 *              mg_color_matrix) chosen the same way from the weights  w_c = sum_{good h} |J_c,h|^2.
 * A selection output needs its random-number input and vice versa (MG_EINVAL otherwise).
 * ws_bytes must be >= mg_workspace_bytes_ex(p, nevt, d_selcol != NULL): the colour selection reads the jamps buffer, which
 * the MG_DIAG_THREAD kernel with MG_CS_FUSED does not otherwise write. */
int mg_sigma_batch_ex(mg_process* p, const double* d_momenta, int nevt, const double* d_alphas, const double* d_rndhel,
                      const double* d_rndcol, double* d_me, int* d_selhel, int* d_selcol, void* d_workspace, size_t ws_bytes,
                      void* cuda_stream);
size_t mg_workspace_bytes_ex(const mg_process* p, int nevt, int want_selcol);

/* Same from HOST buffers (pinned memory recommended): copies h_momenta to an internal device buffer, runs the
 * batch, copies me back, synchronises.  The library allocates and owns the device buffers it needs here. */
int mg_sigma_batch_host(mg_process* p, const double* h_momenta, int nevt, double* h_me);

/* Per-helicity contributions of the last mg_sigma_batch still held in the workspace:
 * copies me_h[ngood][nevt] (already divided by denom) to d_out (DEVICE).  For tests. */
int mg_last_helicity_terms(mg_process* p, int nevt, const void* d_workspace, double* d_out, void* cuda_stream);

/* Device time (ms, CUDA events on the caller's stream) of the stages of the last mg_sigma_batch when option
 * "timing" = 1: [0] diagram kernels, [1] colour sum (0 when fused), [2] helicity sum.  Synchronises. */
int mg_last_stage_ms(mg_process* p, float ms[3]);

/* Number of kernels the last mg_sigma_batch launched (diagram + colour-sum + helicity-sum kernels). */
int mg_last_launch_count(const mg_process* p, int* launches);

/* The same batch for callers that cannot allocate device memory (code under CUDA-graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc).  Only for "gg_ttxgggg", the process whose diagram kernel needs scratch memory: here the
 * scratch is a file-scope static __device__ array of 26 MiB inside the library (8 persistent CTAs' worth; every GPU that
 * loads the library holds it until the process exits) instead of the handle's own areas, so the call makes no cudaMalloc /
 * cudaFree / allocating library call and does not synchronise.  Inputs, output and workspace are the caller's, as in
 * mg_sigma_batch (ws_bytes >= mg_workspace_bytes(p, nevt)).  Limits: nevt <= MG_NOALLOC_MAX_EVENTS, else MG_EINVAL and nothing
 * is launched; a good-helicity list must already be installed (mg_helicity_filter / mg_set_good_helicities), else MG_ESTATE;
 * any other process -> MG_EINVAL.  Throughput is that of 8 CTAs (about 1/18 of the GPU).  ALL calls, from every handle of the
 * process, share the one array: calls that may overlap on the GPU (different streams) race on it -- serialise them.  The
 * array keeps the previous call's contents; the kernel writes every word before reading it, nothing needs clearing.
 * Results are bit-identical to mg_sigma_batch's. */
#define MG_NOALLOC_MAX_EVENTS 256
int mg_sigma_batch_noalloc(mg_process* p, const double* d_momenta, int nevt, double* d_me, void* d_workspace,
                           size_t ws_bytes, void* cuda_stream);

/* Stand-alone colour sum over rows of jamps already in DEVICE memory, layout [2][ncolor][nrows] (re block,
 * im block) of the precision's colour-sum type (fp64 for MG_FP64, fp32 otherwise):
 *   d_out[r] = sum_ij (Re J_i C_ij Re J_j + Im J_i C_ij Im J_j),  C = integer numerators (denominator NOT applied).
 * impl = MG_CS_FUSED runs the scalar-ALU triangular kernel, MG_CS_TENSOR the tensor-core kernel.
 * "gg_ttxgggg" (720 colours): MG_CS_TENSOR in MG_FP64 only (the tcgen05 kernel of that size reads the operand layout the
 * diagram kernel writes, not this one; there is no scalar kernel): anything else -> MG_ECUDA "invalid argument". */
int mg_color_sum(mg_process* p, int impl, const void* d_jamps, long nrows, double* d_out, void* cuda_stream);

/* Copy the integer colour matrix numerators [ncolor*ncolor] and the common denominator to HOST memory. */
int mg_color_matrix(const mg_process* p, int* h_numerators, int* denominator);

/* Micro-benchmarks for roofline denominators (bench.py): kind 0 = fp64 FMA, 1 = fp32 FMA, 2 = DMMA (mma.sync
 * m8n8k4 f64), 3 = tcgen05 kind::tf32.  Returns achieved TFLOP/s in *tflops.  Synchronous. */
int mg_measure_peak(int device, int kind, double* tflops);

const char* mg_last_error(const mg_process* p);
void mg_destroy(mg_process* p);

#ifdef __cplusplus
}
#endif
#endif /* MG5_B200_H */
