/*
 * ttn.h -- C ABI of the B200 tropical tensor-network sweep (libttn.so).
 *
 * The library contracts the tropical tensor network of an L x L open-boundary Ising (q = 2)
 * or 3-state Potts (q = 3) spin glass as a row-by-row transfer sweep in the paper's circuit
 * picture (Fig. 1b; App. A (A2)-(A4) PAPER.md:240-252): a state vector of
 * q^L tropical numbers (Eq. (2)) -- or counting tuples (x, n) (Eq. (4)
 * PAPER.md:78-83) -- goes through every row; a final (+)-reduction gives -E0
 * and the ground-state degeneracy.  A checkpointed backward pass returns one
 * ground-state configuration ("caching intermediate contraction results and backtracking",
 * PAPER.md:97; footnote [49] PAPER.md:201 for ties).
 *
 * Problem statement (Eq. (1)):
 *     E(sigma) = - sum_<ij> J_ij sigma_i sigma_j - sum_i h_i sigma_i ,   sigma_i = +-1
 *   site (r,c), r,c in [0,L);  Jh[r][c] (c < L-1) couples (r,c)-(r,c+1);  Jv[r][c] (r < L-1)
 *   couples (r,c)-(r+1,c);  h[r][c] is the field on (r,c).
 *   Potts (App. C, in BASELINE.json's reading):
 *     E(t) = - sum_<ij> J_ij delta(t_i, t_j),  t_i in {0,1,2},  no fields.
 *
 * Memory spaces.  Couplings and results are HOST pointers (they are O(L^2) numbers);
 * `workspace` is a DEVICE pointer owned by the caller (at least ttn_workspace_bytes(...)
 * bytes, 256-byte aligned), `stream` is a cudaStream_t passed as void* (NULL = default
 * stream).  The library allocates no device memory; its process-wide state is a mutex-guarded
 * memo of searched Potts pass schedules (a pure function of L) and, for ttn_sweep_energy_noalloc
 * only, the built-in scratch array with its per-device address table (see that call).  The TTN_DEBUG_*
 * environment switches are test hooks: they are ignored unless TTN_ENABLE_DEBUG=1 is also set (the
 * test suite sets it), are read once per entry point, and a plan keeps the values it was created with.  Every step of the path runs in the library's own sm_100a kernels.  There
 * is NO CPU fallback: without a CUDA device every compute call returns TTN_ECUDA.
 *
 * h = 0 (NULL or all zero): Eq. (1) is invariant under the global flip sigma -> -sigma, and so is
 * every intermediate state of the sweep; ttn_sweep_energy[_i16], ttn_sweep_count and ttn_ground_config then store only the
 * half of the state vector with column 0 up (2^(L-1) elements) and apply the column-0 gates as a
 * pairing of every element with its complement -- half the memory, bytes and arithmetic,
 * identical results, the degeneracy being twice the half's count.  Any
 * non-zero field selects the full-state sweep.
 *
 * Layouts (row-major, batch-major):  Jh[batch][L][L-1], Jv[batch][L-1][L], h[batch][L][L]
 * (h may be NULL = all zero), E0[batch], degeneracy[batch], sigma[batch][L][L] (+1 / -1).
 *
 * Numerics.  State elements are f32 (Tropical<f32>); degeneracy counts are f64
 * (CountingTropical<f32,f64>): exact below 2^53, correctly rounded sums above.  Ties in
 * Eq. (4) are exact IEEE equality on f32, meaningful for integer-valued couplings.
 * E0 is returned as the ground-state ENERGY (the sweep yields -E0); -0.0 is normalised to
 * +0.0.  Under degeneracy sigma is one ground state (lowest state index wins ties).
 *
 * Errors.  Every function returns a ttn_status; nothing throws or aborts.
 * ttn_last_error() gives a thread-local message for the last non-OK status.
 */
#ifndef TTN_H_
#define TTN_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    TTN_OK = 0,
    TTN_EINVAL = 1,        /* NULL pointer, L < 1, batch < 1, non-finite coupling, bad q/mode   */
    TTN_EUNSUPPORTED = 2,  /* L beyond the limits below, or the device is not sm_100           */
    TTN_ENOMEM = 3,        /* workspace_bytes smaller than ttn_workspace_bytes(...)            */
    TTN_ECUDA = 4          /* a CUDA call failed / no device; see ttn_last_error()             */
} ttn_status;

typedef enum {
    TTN_TROPICAL_F32 = 0,      /* Eq. (2): x (+) y = max, x (.) y = x + y                      */
    TTN_COUNTING_F32_F64 = 1,  /* Eq. (4): (x, n) tuples, n summed on exact ties               */
    TTN_TROPICAL_I16 = 2       /* Eq. (2) on 16-bit integers: integer-valued couplings only, the
                                  paper's own element type for +-J           */
} ttn_semiring;

/* Limits: Ising tropical L <= 34, Ising counting L <= 32, Potts L <= 20 (index fits 32 bits);
   ttn_ground_config L <= 32: L checkpoints of 2^L f32 each up to L = 28, ~2 sqrt(L) of them with a
   re-sweep of every segment in the backward pass beyond; the workspace at L = 32 is
   208 GiB with fields (12 checkpoint buffers + the state; beyond one B200) and 104 GiB for h = 0
   (ttn_workspace_bytes_h0). */

/* Bytes of device workspace needed.  q = 2 (Ising) or 3 (Potts).  Returns 0 on bad arguments.
   The size covers any field h.  ttn_workspace_bytes_h0 is the (smaller) size that suffices when the
   caller will pass h = NULL or an all-zero h (the flip-reduced half-state, see the top of this file);
   at L = 32, ttn_ground_config fits one B200 only in that case. */
size_t ttn_workspace_bytes(int q, int L, ttn_semiring mode, int batch, int want_config);
size_t ttn_workspace_bytes_h0(int q, int L, ttn_semiring mode, int batch, int want_config);

/* ---- one-call host API (upload + sweep + read-back, synchronises `stream`) -------------- */

/* Ground-state energy, Tropical<f32> sweep. */
ttn_status ttn_sweep_energy(int L, const float* Jh, const float* Jv, const float* h, int batch,
                            void* workspace, size_t workspace_bytes, void* stream,
                            double* E0 /*[batch]*/);

/* Same result as ttn_sweep_energy, computed in Tropical<i16> (two state elements per 32-bit word,
   packed add-max): half the state (2^L x 2 bytes) and twice the update rate.  EXACT, and only for
   integer-valued couplings with sum|Jh| + sum|Jv| + sum|h| <= 8000 per instance (every
   intermediate then fits 16 bits); anything else returns TTN_EINVAL.  L < 13 runs the f32 path. */
ttn_status ttn_sweep_energy_i16(int L, const float* Jh, const float* Jv, const float* h, int batch,
                                void* workspace, size_t workspace_bytes, void* stream,
                                double* E0 /*[batch]*/);

/* Ground-state energy and degeneracy, CountingTropical sweep (Eq. (4)). */
ttn_status ttn_sweep_count(int L, const float* Jh, const float* Jv, const float* h, int batch,
                           void* workspace, size_t workspace_bytes, void* stream,
                           double* E0 /*[batch]*/, double* degeneracy /*[batch]*/);

/* Ground-state energy and one ground-state configuration: forward sweep with row-boundary
   checkpoints C_r, backward argmax pass (stands in for App. B). */
ttn_status ttn_ground_config(int L, const float* Jh, const float* Jv, const float* h, int batch,
                             void* workspace, size_t workspace_bytes, void* stream,
                             double* E0 /*[batch]*/, int8_t* sigma /*[batch][L][L]*/);

/* 3-state Potts variants (App. C): 3x3 max-plus gates, state 3^L. */
ttn_status ttn_potts3_sweep_energy(int L, const float* Jh, const float* Jv, int batch,
                                   void* workspace, size_t workspace_bytes, void* stream,
                                   double* E0 /*[batch]*/);
ttn_status ttn_potts3_sweep_count(int L, const float* Jh, const float* Jv, int batch,
                                  void* workspace, size_t workspace_bytes, void* stream,
                                  double* E0 /*[batch]*/, double* degeneracy /*[batch]*/);

/* ---- for callers that cannot allocate device memory --------------------------------------
 * ttn_sweep_energy (same sweep, same kernels, same result: PAPER.md:103-118) without the `workspace`
 * argument.  It is meant for code that has no way to get device memory of its own -- a plug-in or
 * callback inside a host application whose memory pool already owns the whole GPU (a raw cudaMalloc
 * there fails and the plug-in has no handle to the pool), or a loop that must not run into the
 * device-wide synchronisation that cudaMalloc / cudaFree imply.  The scratch memory is an array of
 * TTN_NOALLOC_SCRATCH_BYTES that is part of the library image: every GPU that loads libttn.so holds
 * that much from load to process exit, whether or not this function is ever called.  The call
 * allocates and frees no device memory (the pass schedule lives on the host heap for the duration
 * of the call; leave the TTN_DEBUG_TIMING test switch unset, it creates CUDA events).
 *   Limit: the workspace the ordinary call would need, ttn_workspace_bytes(2, L, TTN_TROPICAL_F32,
 *     batch, 0) -- or ttn_workspace_bytes_h0(...) when h is NULL / all zero -- must fit the array:
 *     batch 1 up to L = 20 with a field and L = 21 without; small lattices in batches (e.g. 14
 *     instances of 16 x 16 with fields).  Anything larger returns TTN_EUNSUPPORTED with a message
 *     that states both sizes, before any CUDA call.
 *   First call on a device: looks up the array's address on the CURRENT device
 *     (cudaGetSymbolAddress) and keeps it; make that first call outside any stream capture.
 *   Sharing: all calls on one device, from any thread or stream, use the SAME array.  Calls that
 *     overlap on the GPU race on it and give garbage; calls on one stream, or otherwise ordered, are
 *     safe.  The array keeps what the last call left, and no call depends on it: every byte a sweep
 *     reads it has written first, so nothing needs clearing between calls.
 *   Jh, Jv, h, E0 are HOST pointers with the layouts above; the call synchronises `stream`. */
#define TTN_NOALLOC_SCRATCH_BYTES 4718592 /* 4.5 MiB */
ttn_status ttn_sweep_energy_noalloc(int L, const float* Jh, const float* Jv, const float* h, int batch,
                                    void* stream, double* E0 /*[batch]*/);

/* ---- chimera graph (Fig. 2) -------------------------
 * +-J (any integer couplings), no field, on M x N unit cells of K_{4,4}: cell (r, c) holds a
 * vertical group v[0..4) and a horizontal group u[0..4);
 *   K [M][N][4][4]  K[r][c][k][l] couples v_k and u_l of the same cell,
 *   Jv[M-1][N][4]   couples v_k of (r, c) with v_k of (r+1, c)   (may be NULL when M = 1),
 *   Jh[M][N-1][4]   couples u_l of (r, c) with u_l of (r, c+1)   (may be NULL when N = 1),
 * energy as Eq. (1) with h = 0.  All three are HOST pointers, row-major float32.  The sweep runs
 * column by column at the level of single spins in Tropical<i16> (the paper's Int16):
 * a state of 2^(4M+4) int16 elements (the 4M horizontal spins of the column front and a 4-spin
 * ancilla for the vertical group), one HBM pass per unit cell -- for M <= 3; for M >= 4 the state is
 * the paper's 16^M column front, 2^(4M) int16 elements (M = 8: 8 GiB), swept with three gate-row
 * passes and one vertical-chain pass per column of cells (csrc/ttn_chimera2.cuh).  Exact; couplings
 * must be integer-valued with sum |J| <= 8000 (every intermediate then fits 16 bits), else
 * TTN_EINVAL: for +-J couplings that bounds the number of edges, i.e. N <= 42 at M = 8 (184 edges
 * per column of 8 cells), whatever the structural limits M <= 8, N <= 64 (beyond those:
 * TTN_EUNSUPPORTED).  `workspace` is a DEVICE pointer of at least
 * ttn_chimera_workspace_bytes(M, N) bytes (0 = unsupported size); E0 receives the ground-state
 * energy; the call synchronises `stream`. */
size_t ttn_chimera_workspace_bytes(int M, int N);
ttn_status ttn_chimera_sweep_energy_i16(int M, int N, const float* K, const float* Jv, const float* Jh,
                                        void* workspace, size_t workspace_bytes, void* stream,
                                        double* E0 /*[1]*/);

/* Ground-state energy AND degeneracy on the chimera graph (CountingTropical, Eq. (4) PAPER.md:78-83;
 * the residual entropies of PAPER.md:128, Fig. 3): same arguments and conventions as
 * ttn_chimera_sweep_energy_i16, elements (x f32, n f64), 12 bytes per state of the 16^max(M,3) column
 * front (M = 8: 48 GiB).  Couplings must be integer-valued (exact f32 sums and exact ties), else
 * TTN_EINVAL.  degeneracy is exact below 2^53 and a correctly rounded f64 product / sum above. */
size_t ttn_chimera_count_workspace_bytes(int M, int N);
ttn_status ttn_chimera_sweep_count(int M, int N, const float* K, const float* Jv, const float* Jh,
                                   void* workspace, size_t workspace_bytes, void* stream,
                                   double* E0 /*[1]*/, double* degeneracy /*[1]*/);

/* ---- split API: upload once, launch asynchronously, read later ---------------------------
 * The one-call functions above are ttn_plan_create + ttn_plan_launch + ttn_plan_read +
 * ttn_plan_destroy.  A plan holds the host-side pass schedule (which gates
 * and diagonal terms each HBM pass applies) and the addresses of its tables inside
 * `workspace`; the workspace must stay alive and untouched while the plan is in use.
 *   ttn_plan_create : validates, plans, copies couplings host->device on `stream` (async).
 *   ttn_plan_launch : enqueues every kernel of one whole sweep on `stream`; does not
 *                     synchronise; results stay in the workspace.  May be called repeatedly.
 *   ttn_plan_read   : device->host copy of the results of the last launch; synchronises.
 *                     Pointers that do not apply to the plan's call kind must be NULL.      */
typedef struct ttn_plan ttn_plan;
typedef enum {
    TTN_CALL_ENERGY = 0, TTN_CALL_COUNT = 1, TTN_CALL_CONFIG = 2, TTN_CALL_ENERGY_I16 = 3,
    /* TTN_CALL_ENERGY with the flip-reduced half-state REQUIRED: TTN_EINVAL when h != 0 (lattices with
       L < 14 run the plain sweep).  TTN_CALL_ENERGY selects it by itself when h = 0; this kind exists
       for ttn_plan_describe and for tests. */
    TTN_CALL_ENERGY_Z2 = 4,
    TTN_CALL_COUNT_Z2 = 5,      /* the same for TTN_CALL_COUNT (L < 12 runs the plain sweep) */
    TTN_CALL_ENERGY_I16_Z2 = 6, /* the same for TTN_CALL_ENERGY_I16 (L < 15 runs the plain i16 sweep) */
    TTN_CALL_CONFIG_Z2 = 7      /* the same for TTN_CALL_CONFIG: checkpoints are half-states (L < 14: plain) */
} ttn_call;

ttn_status ttn_plan_create(int q, int L, ttn_call call, const float* Jh, const float* Jv,
                           const float* h, int batch, void* workspace, size_t workspace_bytes,
                           void* stream, ttn_plan** plan);
ttn_status ttn_plan_launch(ttn_plan* plan, void* stream);
ttn_status ttn_plan_read(ttn_plan* plan, void* stream, double* E0, double* degeneracy,
                         int8_t* sigma);
void ttn_plan_destroy(ttn_plan* plan);

/* Introspection (host only, no CUDA calls). */
int ttn_plan_num_launches(const ttn_plan* plan);   /* kernels enqueued by one ttn_plan_launch   */
int ttn_plan_num_passes(const ttn_plan* plan);     /* HBM passes over the state among them      */
/* State-vector elements stored per instance: q^L, or 2^(L-1) when the plan uses the h = 0 flip
   reduction (see the top of this file). */
unsigned long long ttn_plan_state_elements(const ttn_plan* plan);
/* Writes a text description of the pass schedule for (q, L, call) -- one line per pass and
   one per op -- into buf (NUL-terminated, truncated to n).  Returns the untruncated length,
   or -1 on bad arguments.  Needs no device: used by the CPU-side schedule validator.          */
long ttn_plan_describe(int q, int L, ttn_call call, char* buf, size_t n);

const char* ttn_last_error(void);   /* thread-local, static storage */
int ttn_version(void);

#ifdef __cplusplus
}
#endif
#endif /* TTN_H_ */
