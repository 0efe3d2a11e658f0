// rcg_internal.h -- shared declarations of the library's translation units (not installed).
// Data model of the generated per-class sources (csrc/gen/eri_<la><lb><lc><ld>.cu).
#ifndef RCG_INTERNAL_H
#define RCG_INTERNAL_H
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/rcg.h"

// Device view of a basis handle (all pointers DEVICE).
struct RcgBasisDev {
    const double *centers;    // [nshell][3]
    const int32_t *prim_off;  // [nshell+1]
    const double *exps;       // [nprim]
    const double *coefs;      // [nprim]
    const int32_t *shell_l;   // [nshell]
    const double *boys;       // Boys Taylor grid [RCG_BOYS_NROW][RCG_BOYS_NCOL]
    int nshell;
};

// One launch of a class kernel.  perm: canonical position k takes the caller's quartet column
// perm[k]; ostride[k]: stride (in doubles) of canonical spherical index k in the caller's layout.
struct RcgLaunch {
    RcgBasisDev basis;
    const int32_t *quartets;  // [n][4]
    int64_t n;
    double *out;
    int64_t out_stride;       // doubles per quartet
    int perm[4];
    int nsph[4];              // 2l+1 of the canonical indices
    int lcan[4];              // angular momenta of the canonical indices
    int kmin[5], kmax[5];     // min / max primitives per shell of each angular momentum in the basis
    int64_t ostride[4];
    double *workspace;
    cudaStream_t stream;
    const unsigned long long *stat;   // DEVICE [2] {padded, real} primitive work of the packed grouping, or nullptr
    struct RcgStatHolder *stat_holder;    // HOST, owned by the API call: lazily allocated device words for `stat` / `stat_reg`
    const unsigned long long *stat_reg;   // DEVICE [2] {padded, real} work of 32 quartets per warp (register tier), or nullptr
    int force_tier;                   // 0, or the tier the caller asked for (rcg_eri_batch_tier)
    // Fock build (rcg_fock_batch): digestion fused into the class kernel; all null / 0 for rcg_eri_batch
    const int32_t *bf_off;            // DEVICE [nshell] first basis function of each shell
    const double *D;                  // DEVICE [nbf][nbf] symmetric density
    double *Jt, *Kt;                  // DEVICE [nbf][nbf], accumulated into
    int nbf;
    int uniform_k4;                   // 1: the caller promises one K4 for the whole list (rcg_eri_batch_uniform): no statistics pass
};

typedef cudaError_t (*RcgLaunchFn)(const RcgLaunch &);

// Table-driven global tier (see gen/emit_global.py for the record formats).  HOST pointers.
struct RcgGlobalTables {
    const uint32_t *vrr_fam; int n_fam;
    const int32_t *lvl_off;  int n_levels;     // families [lvl_off[l], lvl_off[l+1]) are mutually independent
    const int32_t *tslots;                     // slot of the k-th target in level order
    const int32_t *tindex;                     // its index a*nC+c in H
    const int32_t *tgt_off;  int n_targets;    // targets of level l: [tgt_off[l], tgt_off[l+1]), l = 0..n_levels
    int nA, nC;              // bra / ket target components (Cartesian)
    int n_vslots;
    // Phase-2 node programs (level-sorted; see gen/emit_global.py): words, node offsets, level offsets
    const uint32_t *bra_ops; int n_bra_words; const int32_t *bra_noff; int n_bra_nodes; const int32_t *bra_loff; int n_bra_levels;
    int bra_nin; int bra_nslots; const uint16_t *bra_out; int bra_nout;
    const uint32_t *ket_ops; int n_ket_words; const int32_t *ket_noff; int n_ket_nodes; const int32_t *ket_loff; int n_ket_levels;
    int ket_nin; int ket_nslots; const uint16_t *ket_out; int ket_nout;
    const double *consts;    int n_consts;
};

struct RcgClassDesc {
    int l[4];
    int tier;
    long long flops_prim, flops_quartet;
    int vrr_vertices, peaklive;
    RcgGlobalTables g;
    RcgLaunchFn launch;      // specialised (register / warp / block tier) launcher or nullptr
    RcgLaunchFn launch_fock; // kernel with the J/K digestion in its epilogue, or nullptr
    int fock_kind;           // 1: thread-per-quartet kernel (long lists with one K4 only), 2: warp-tier kernel (any list), 0: none
    long long ws_quartet_doubles;   // heavy block tier: workspace doubles per quartet of a chunk (csrc/rcg_sides.h), else 0
};

extern const RcgClassDesc *const rcg_class_table[];
extern const int rcg_class_count;

// pack_stats.cu: enqueue the padding statistics of a packed grouping with Q quartets per warp.  The two result words live
// in a block the API call owns (RcgStatHolder): allocated stream-ordered on the call's stream from the library's memory
// pool on first need, freed stream-ordered by the API after the class's kernels are enqueued -- so a slot can neither be
// shared by two host threads nor recycled under a pending launch on another stream.  which: 0 -> words 0,1 (packed
// grouping), 1 -> words 2,3 (register tier, groups of 32).
struct RcgStatHolder { cudaStream_t stream; unsigned long long *words; };
cudaError_t rcg_pack_stats(const RcgLaunch &a, int Q, int which, const unsigned long long **stat);
cudaError_t rcg_stat_release(RcgStatHolder &h);
cudaError_t rcg_pool_alloc(void **p, size_t bytes, cudaStream_t stream);      // rcg_api.cu: the per-device retained pool

// Per-device facts and one-time kernel preparation, safe for concurrent host threads (atomics; a lost race repeats an
// idempotent call).  rcg_prepare_kernel raises the kernel's dynamic shared-memory limit once per device and returns the SM count.
#include <atomic>
struct RcgOnce { std::atomic<unsigned long long> done{0}; };
cudaError_t rcg_sm_count(int *nsm);
cudaError_t rcg_prepare_kernel(RcgOnce &once, const void *func, size_t smem_bytes, int *nsm);

// rcg_api.cu: record the CUDA error for rcg_last_cuda_error (thread-local) and return RCG_ERR_CUDA
rcg_status rcg_cuda_fail(cudaError_t e);

// tier_global.cu
cudaError_t rcg_global_launch(const RcgClassDesc &d, const RcgLaunch &a);
size_t rcg_global_workspace_bytes(const RcgClassDesc &d, int64_t n);

// eri_grad.cu: first derivatives with respect to the four centres (one class-independent kernel, a block per quartet)
struct RcgGradLaunch {
    RcgBasisDev basis;
    const int32_t *quartets;  // [n][4]
    int64_t n;
    double *out;              // [n][12][2la+1][2lb+1][2lc+1][2ld+1]
    int l[4];                 // the caller's (la, lb, lc, ld); the kernel puts the heavier shell of each pair first
    long long k4max;          // largest number of primitive quartets a quartet of this class can have in the basis, or the caller's promise
    int k4_promised;          // 1: every quartet of the list has k4max primitive quartets (rcg_eri_grad_batch_uniform)
    cudaStream_t stream;
};
bool rcg_grad_supported(const int l[4], size_t *smem_bytes);   // the block's accumulators and tables fit 227 KB, Boys order <= 16
cudaError_t rcg_grad_launch(const RcgGradLaunch &a);

#define RCG_BOYS_TS 36.0     // switch to the asymptotic branch (R-BOYS)
#define RCG_BOYS_NROW 289    // T0 = row/8, row = 0..288
#define RCG_BOYS_NCOL 25     // orders 0..24 (L<=16 plus 8 Taylor terms)
extern const double rcg_boys_table_host[RCG_BOYS_NROW * RCG_BOYS_NCOL];

#endif
