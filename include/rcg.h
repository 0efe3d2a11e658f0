/*
 * rcg.h -- C ABI of the B200-native batched HGP electron-repulsion-integral library.
 *
 * What the calls compute (citations are PAPER.md lines of arxiv/paper_2605_10312):
 *   contracted, real-spherical ERIs (ab|cd) of Eq. (1) for a list of shell
 *   quartets of ONE angular class (la lb|lc ld), by the Head-Gordon-Pople pipeline of
 *   Alg. 2:  Gaussian-pair quantities (:80) -> Boys F_m(T) (:69, :273)
 *   -> Obara-Saika vertical recurrence, Eq. (2) (:69-80) -> primitive contraction (:275)
 *   -> horizontal recurrence, Eq. (3) (:82-87) fused with the stepwise Cartesian->spherical
 *   transform, Eqs. (8)-(16) (:183-231).  rcg_eri_batch writes the integrals to an output buffer;
 *   rcg_fock_batch digests them into J/K instead, as the paper does (:259, :267, :291);
 *   rcg_eri_grad_batch writes their first derivatives with respect to the four centres (:299).
 *
 * Conventions: primitives are UNNORMALISED Cartesian Gaussians and
 * coefficients are used as given (R-PRIM); spherical components are rows m=-l..l of the
 * Racah-normalised real solid harmonics (R-SPH), p shells therefore (y,z,x); FP64 only;
 * no screening and no symmetry factors inside the calls.
 *
 * Memory: every pointer is tagged HOST or DEVICE below.  The caller owns every buffer; the
 * handle owns only its private device copies (shell data, Boys grid) and frees them in
 * rcg_basis_destroy.  Streams are passed as void* (a cudaStream_t; NULL = default stream).
 * Errors: every call returns an rcg_status (0 = RCG_OK, <0 = error); nothing throws, aborts
 * or prints.  There is no CPU fallback: without a CUDA device the calls return RCG_ERR_CUDA.
 */
#ifndef RCG_H
#define RCG_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rcg_basis rcg_basis; /* opaque */
typedef int rcg_status;

#define RCG_OK 0
#define RCG_ERR_INVALID_ARG (-1)         /* null pointer, negative count, l > RCG_LMAX, misaligned list */
#define RCG_ERR_UNSUPPORTED_CLASS (-2)   /* no kernel was generated for this angular class */
#define RCG_ERR_WORKSPACE_TOO_SMALL (-3) /* workspace_bytes < rcg_eri_workspace_bytes(...) */
#define RCG_ERR_CUDA (-4)                /* CUDA runtime failure; see rcg_last_cuda_error */
#define RCG_ERR_CLASS_MISMATCH (-5)      /* rcg_validate_batch: a listed shell has the wrong l */
#define RCG_ERR_STATIC_SCRATCH_LIMIT (-6) /* rcg_eri_batch_static: the batch needs more than RCG_STATIC_SCRATCH_BYTES of scratch */

#define RCG_LMAX 4
#define RCG_KMAX 45                      /* primitives per shell (the kernels decode a primitive-quartet index < 2^22) */

/* Tier a class was generated for (PAPER.md:251-257 tiers, re-derived for sm_100a). */
#define RCG_TIER_REGISTER 1 /* one thread per quartet, recurrence graph fully in registers        */
#define RCG_TIER_WARP 2     /* lane = bra Cartesian component, cross terms through shared memory   */
#define RCG_TIER_GLOBAL 3   /* table-driven, intermediates in an interleaved global scratch (:265) */
#define RCG_TIER_BLOCK 4    /* one thread block per quartet: thread = bra component, ket chains in */
                            /* registers, chain heads in shared memory ((fd|pp) ... (gg|gg))        */

/* Build a basis handle.  Input arrays are HOST pointers and are copied; they may be freed
 * on return.  shell_l[nshell] in 0..RCG_LMAX; shell_prim_offset[nshell+1] CSR offsets into
 * exps/coefs (nprim = last offset), 1..RCG_KMAX primitives per shell; exps > 0; coefs carry ALL normalisation (R-PRIM);
 * centers[nshell][3] in Bohr (Alg. 2 line 1).  The device copies are made on
 * `stream`; the handle is immutable afterwards and may be used from several streams. */
rcg_status rcg_basis_create(rcg_basis **out, int nshell, int nprim, const int32_t *shell_l,
                            const int32_t *shell_prim_offset, const double *exps,
                            const double *coefs, const double *centers, void *stream);
rcg_status rcg_basis_destroy(rcg_basis *b);

/* Scratch the class needs for `nquartet` quartets: 0 for the register, warp and slab-block kernels with Phase 2 inside; for the
 * block-tier classes with Phase 2 in the side kernels (every class with a g shell, light-ket (fd|xx) / (ff|xx)) the hand-over buffer of
 * one chunk, bytes per quartet x min(nquartet, chunk), where a chunk is a whole number of waves of the CURRENT device's SM count
 * (so the figure depends on the device that is current; it must be the handle's).  HOST out. */
rcg_status rcg_eri_workspace_bytes(const rcg_basis *b, int la, int lb, int lc, int ld,
                                   int64_t nquartet, size_t *bytes);

/* The hot path (Alg. 2, with a plain store instead of line 10's scatter).
 *   quartets  DEVICE int32[nquartet][4], shell indices (a,b,c,d), 16-byte aligned; shell a
 *             must have angular momentum la, b lb, c lc, d ld (not checked here; see
 *             rcg_validate_batch).  Repeated indices are legal.
 *   out       DEVICE double[nquartet][2la+1][2lb+1][2lc+1][2ld+1], C order, OVERWRITTEN.
 *   workspace DEVICE scratch of at least rcg_eri_workspace_bytes bytes (may be NULL if 0).
 * Any (la,lb,lc,ld) with l <= RCG_LMAX = 4 is accepted (all 120 pair-canonical classes are generated): non-canonical orders are mapped
 * onto the generated canonical class (la>=lb, lc>=ld, (la,lb)>=(lc,ld)) by
 * (ab|cd)=(ba|cd)=(ab|dc)=(cd|ab) and written in the CALLER's index order.
 * Asynchronous: enqueues on `stream` and returns; nquartet == 0 is a no-op. */
rcg_status rcg_eri_batch(const rcg_basis *b, int la, int lb, int lc, int ld,
                         const int32_t *quartets, int64_t nquartet, double *out,
                         void *workspace, size_t workspace_bytes, void *stream);

/* rcg_eri_batch for a list whose quartets ALL have the same number of primitive quartets K4 = Ka Kb Kc Kd -- the caller's
 * promise (e.g. the batches of a screened pass that buckets its pair lists by contraction depth).  The launcher then skips
 * the device-side statistics pass that chooses between the thread-per-quartet, packed and one-quartet-per-warp kernels of the
 * light classes and takes the kernel made for even lists.  Same results; a broken promise only costs speed. */
rcg_status rcg_eri_batch_uniform(const rcg_basis *b, int la, int lb, int lc, int ld,
                                 const int32_t *quartets, int64_t nquartet, double *out,
                                 void *workspace, size_t workspace_bytes, void *stream);

/* rcg_eri_batch for callers that may not allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc): the
 * scratch of the launch lives in a device array of RCG_STATIC_SCRATCH_BYTES (32 MiB) that is part of the library image -- every GPU
 * that loads the library holds it until the process exits -- and the call makes no cudaMalloc / cudaFree / allocating library call.
 * Only for the classes whose kernels USE scratch (block-tier classes with Phase 2 in the side kernels: every class with a g shell and
 * the light-ket (fd|xx), (ff|xx) classes; rcg_eri_workspace_bytes > 0); any other class returns RCG_ERR_UNSUPPORTED_CLASS (it needs
 * no scratch: rcg_eri_batch with a NULL workspace allocates nothing either).  A batch whose scratch (bytes per quartet of the class x
 * nquartet) exceeds the array returns RCG_ERR_STATIC_SCRATCH_LIMIT and launches nothing; rcg_eri_batch_static_max_quartets gives the
 * largest nquartet the class admits ((gg|gg): 127; (gs|ss): 174,762).  Same arguments, results and asynchrony as rcg_eri_batch.
 * ALL calls share the one array (it keeps the last call's contents; nothing in it needs clearing): calls that overlap on the GPU --
 * different streams without an ordering between them -- race; calls on one stream are safe. */
#define RCG_STATIC_SCRATCH_BYTES (32 << 20)
rcg_status rcg_eri_batch_static(const rcg_basis *b, int la, int lb, int lc, int ld,
                                const int32_t *quartets, int64_t nquartet, double *out, void *stream);
rcg_status rcg_eri_batch_static_max_quartets(const rcg_basis *b, int la, int lb, int lc, int ld, int64_t *max_quartets);

/* Same computation with HOST quartets and HOST out (pinned or pageable): copies the list
 * to the device, runs rcg_eri_batch chunk by chunk (at least 32 MB of output per chunk), copies
 * each chunk back on an internal second stream while the next one is computed (the overlap needs
 * pinned memory), and synchronises `stream`.  Device staging comes from a stream-ordered memory
 * pool the library keeps per device (its memory is retained between calls and released at
 * process exit); nothing of it is visible to the caller. */
rcg_status rcg_eri_batch_host(const rcg_basis *b, int la, int lb, int lc, int ld,
                              const int32_t *quartets_host, int64_t nquartet, double *out_host,
                              void *stream);

/* Same computation on a chosen tier: RCG_TIER_GLOBAL (table-driven, every class has it, scratch = the interleaved slot buffer of
 * the independent cross-check of the specialised tiers at sizes the CPU oracle cannot reach), the class's own tier, or
 * RCG_TIER_WARP for a register-tier class; any other combination returns RCG_ERR_UNSUPPORTED_CLASS.  tier = 0: rcg_eri_batch. */
rcg_status rcg_eri_batch_tier(const rcg_basis *b, int tier, int la, int lb, int lc, int ld,
                              const int32_t *quartets, int64_t nquartet, double *out,
                              void *workspace, size_t workspace_bytes, void *stream);
rcg_status rcg_eri_workspace_bytes_tier(const rcg_basis *b, int tier, int la, int lb, int lc,
                                        int ld, int64_t nquartet, size_t *bytes);

/* Debug pass: DEVICE quartets; synchronises; RCG_ERR_CLASS_MISMATCH if any listed shell index
 * is out of range or has the wrong angular momentum. */
rcg_status rcg_validate_batch(const rcg_basis *b, int la, int lb, int lc, int ld,
                              const int32_t *quartets, int64_t nquartet, void *stream);

/* Screened pass helpers (BASELINE.json configs 3 and 5: unique quartets with Schwarz bound above a
 * threshold, batched by angular class; reading R-SCHWARZ in DESIGN.md).  List logic only.
 * rcg_schwarz_from_blocks: blocks = DEVICE double[n][dim][dim], the (ab|ab) blocks rcg_eri_batch wrote for
 *   the quartets (a,b,a,b) with dim = (2la+1)(2lb+1); Q[i] = sqrt(max_k |blocks[i][k][k]|), DEVICE double[n].
 * rcg_quartets_from_pairs: bra_pairs / ket_pairs = DEVICE int32[.][2] shell pairs (8-byte aligned), the ket
 *   list sorted by decreasing Q; offs = DEVICE int64[nbra+1], exclusive prefix sum of the number of
 *   surviving ket pairs (a prefix of the sorted ket list) per bra pair.  Writes rows
 *   offs[i]-offs[i0]+j = (bra_pairs[i], ket_pairs[j]), i in [i0,i1), j < offs[i+1]-offs[i], into
 *   quartets (DEVICE int32[offs[i1]-offs[i0]][4], 16-byte aligned, caller-sized).  Asynchronous. */
rcg_status rcg_schwarz_from_blocks(const double *blocks, int64_t n, int dim, double *Q, void *stream);
rcg_status rcg_quartets_from_pairs(const int32_t *bra_pairs, const int32_t *ket_pairs, const int64_t *offs,
                                   int64_t i0, int64_t i1, int32_t *quartets, void *stream);

/* J/K digestion (Alg. 2 line 10 at :283):
 *   J_mn = sum_ls D_ls (mn|ls),   K_mn = sum_ls D_ls (ml|ns)      over spherical basis functions,
 * from the blocks rcg_eri_batch wrote for a list of UNIQUE shell quartets of class (la lb|lc ld) in the order
 * of the call (one representative per 8-fold symmetry orbit: the scale factors 1/2 for a == b, c == d and
 * (a,b) == (c,d) are applied inside).  All pointers DEVICE.  integrals = double[nquartet][2la+1][2lb+1][2lc+1][2ld+1];
 * shell_bf_offset = int32[nshell], first basis function of each shell (functions m = -l..l of a shell are
 * consecutive); D = double[nbf][nbf], SYMMETRIC; Jt, Kt = double[nbf][nbf], ACCUMULATED into (atomicAdd; zeroed
 * by the caller before the first batch).  After the last batch rcg_jk_finish replaces Jt by J = Jt + Jt^T and
 * Kt by K = Kt + Kt^T; only these sums are defined (a kernel may add a contribution to Kt[c][a] instead of Kt[a][c]).
 * Asynchronous on `stream`. */
rcg_status rcg_jk_digest(int la, int lb, int lc, int ld, const int32_t *quartets, int64_t nquartet,
                         const double *integrals, const int32_t *shell_bf_offset, const double *D,
                         double *Jt, double *Kt, int nbf, void *stream);
rcg_status rcg_jk_finish(double *Jt, double *Kt, int nbf, void *stream);

/* Fock build of one batch with the digestion FUSED: the integrals of the listed unique quartets are contracted with D into
 * Jt, Kt (same meaning, scale factors and rcg_jk_finish as rcg_jk_digest) without a trip through HBM.  Classes of the register
 * tier on lists of at least 8,192 quartets with uniform_k4 != 0 (the caller's promise that every quartet has the same number
 * of primitive quartets): the digestion runs in the class kernel's epilogue, from registers, by atomicAdd ("inline
 * atomicAdd scatter ... zero global intermediates").  Everything else: the class kernel writes chunks of at most 1 GiB into
 * `workspace`, overwritten in place chunk after chunk, and the buffered digestion reads them.  (la,lb,lc,ld) must be in CANONICAL order (la >= lb, lc >= ld, (la,lb) >= (lc,ld)) -- the order a
 * screened pass over unique quartets produces; RCG_ERR_INVALID_ARG otherwise.  quartets DEVICE int32[n][4], 16-byte aligned;
 * workspace DEVICE, at least rcg_fock_workspace_bytes (0 for the fused kernels).  Asynchronous on `stream`. */
rcg_status rcg_fock_workspace_bytes(const rcg_basis *b, int la, int lb, int lc, int ld, int64_t nquartet,
                                    int uniform_k4, size_t *bytes);
rcg_status rcg_fock_batch(const rcg_basis *b, int la, int lb, int lc, int ld, const int32_t *quartets,
                          int64_t nquartet, int uniform_k4, const int32_t *shell_bf_offset, const double *D,
                          double *Jt, double *Kt, int nbf, void *workspace, size_t workspace_bytes, void *stream);

/* First derivatives of the integrals with respect to the four shell centres ("first-derivative
 * variants", :401; the scheme of the Head-Gordon-Pople reference): with [a| a primitive Cartesian Gaussian of
 * exponent alpha on centre A,  d/dA_i [a| = 2 alpha [a + 1_i| - a_i [a - 1_i|  (reading R-GRAD in DESIGN.md), the raised and
 * lowered integrals by Eq. (2), (3), contraction Eq. (1) and the transform Eq. (8) as in rcg_eri_batch.
 *   quartets  DEVICE int32[nquartet][4], 16-byte aligned; shell of column k must have angular momentum (la,lb,lc,ld)[k].
 *   out       DEVICE double[nquartet][12][2la+1][2lb+1][2lc+1][2ld+1], C order, OVERWRITTEN; derivative index 3 * k + i for the
 *             centre of quartet COLUMN k (a, b, c, d) and axis i (x, y, z).  Columns are differentiated one by one: if one shell
 *             stands in two columns, the derivative with respect to its centre is the sum of the two column blocks.  The d block
 *             is minus the sum of the other three (translational invariance).
 * One class-independent kernel template: a thread block per quartet with every intermediate in shared memory (light classes: 8 to 64
 * quartets per block; the heaviest: accumulators in a scratch that stays in the L2); any (la,lb,lc,ld) order is
 * accepted (inside, the heavier shell of each pair takes the first position, as in the canonical order of the integral classes: the
 * horizontal recurrence then moves angular momentum DOWN from it; blocks and components are written in the caller's order).
 * Supported (rcg_eri_grad_supported tells, with the shared-memory bytes of a block): the classes whose recurrence buffers fit the
 * 227 KB of a block and whose top Boys order la+lb+lc+ld+2 is at most 16 -- every class of s, p, d shells, all 55 pair-canonical
 * classes of lmax = 3, 111 of the 120 of lmax = 4; the others return RCG_ERR_UNSUPPORTED_CLASS.  Where the accumulators and the
 * buffers of the second phase do not fit beside the recurrence buffers ((fd|fd), (ff|dd), (ff|fd), (ff|ff), most g classes) they live in
 * a scratch of at most 0.6 MB per SM that the call takes from the library's stream-ordered memory pool on `stream` and returns to it
 * stream-ordered after the launch (the pool retains its memory; no synchronisation); every other class uses no scratch and allocates nothing.
 * Asynchronous on `stream`; nquartet == 0 is a no-op. */
rcg_status rcg_eri_grad_batch(const rcg_basis *b, int la, int lb, int lc, int ld, const int32_t *quartets,
                              int64_t nquartet, double *out, void *stream);
rcg_status rcg_eri_grad_supported(int la, int lb, int lc, int ld, int *supported, size_t *smem_bytes); /* HOST outs; smem_bytes may be NULL */
/* rcg_eri_grad_batch for a list whose quartets ALL have k4 = Ka Kb Kc Kd primitive quartets -- the caller's promise (a screened pass that
 * buckets its pair lists by contraction depth).  The light classes have two block organisations: a sub-warp group of 4 to 32 lanes per
 * quartet, many quartets per block (shallow contractions), and eight one-warp primitive groups per quartet (k4 >= 256); without the promise
 * a basis that allows 256 and more primitive quartets in the class gets two launches over the list, each taking its kind of quartet.
 * Same results; a broken promise only costs speed. */
rcg_status rcg_eri_grad_batch_uniform(const rcg_basis *b, int la, int lb, int lc, int ld, const int32_t *quartets,
                                      int64_t nquartet, int64_t k4, double *out, void *stream);

/* Boys function alone (Alg. 2 line 5 at :273; scheme R-BOYS in DESIGN.md):
 * out[i][m] = F_m(T[i]), m = 0..mmax <= 16.  DEVICE T[n], DEVICE out[n][mmax+1]. */
rcg_status rcg_boys(int mmax, const double *T, int64_t n, double *out, void *stream);

/* Static facts the generator recorded for a class (HOST outs, any may be NULL):
 * tier; algorithmic FP64 flops per PRIMITIVE quartet (pair setup + Boys + VRR + contraction)
 * and per CONTRACTED quartet (HRR + stepwise c2s); FMA = 2, MUL/ADD = 1. */
rcg_status rcg_class_info(int la, int lb, int lc, int ld, int *tier,
                          int64_t *flops_per_prim_quartet, int64_t *flops_per_quartet);

/* Number of generated canonical classes, and the i-th one's (la,lb,lc,ld). */
int rcg_num_classes(void);
rcg_status rcg_class_at(int i, int *la, int *lb, int *lc, int *ld);

/* Measurement aid (not on the ERI path): sustained FP64 FMA throughput of the current device in
 * TFLOP/s from a register-only DFMA microbenchmark (about 10 ms); synchronises `stream`.  HOST out. */
rcg_status rcg_fp64_peak_tflops(double *tflops, void *stream);

const char *rcg_status_string(rcg_status s);
int rcg_last_cuda_error(void); /* the cudaError_t of the last RCG_ERR_CUDA on this thread */

#ifdef __cplusplus
}
#endif
#endif /* RCG_H */
