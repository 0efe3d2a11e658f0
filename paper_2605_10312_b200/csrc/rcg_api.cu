// rcg_api.cu -- the C ABI of include/rcg.h: handle management, class canonicalisation, dispatch.
// No arithmetic of the method lives here except rcg_boys' test kernel; see the tier sources.
#include <mutex>
#include <new>
#include <vector>
#include <cstring>
#include "../../include/rcg.h"
#include "rcg_device.cuh"
#include "rcg_sides.h"

struct rcg_basis {
    RcgBasisDev dev;
    void *blob;          // one device allocation holding every array of `dev` except boys
    int kmin[5], kmax[5]; // min / max contraction depth per angular momentum
    int device;          // the device the handle (blob, Boys grid) lives on; every call checks it is current
};

static thread_local int tl_cuda_error = 0;
rcg_status rcg_cuda_fail(cudaError_t e);
static rcg_status cuda_fail(cudaError_t e) { return rcg_cuda_fail(e); }
rcg_status rcg_cuda_fail(cudaError_t e)      // also used by jk_digest.cu, quartet_lists.cu: rcg_last_cuda_error reports THIS error
{
    tl_cuda_error = (int)e;
    return RCG_ERR_CUDA;
}

// ---------------------------------------------------------------- Boys grid (one copy per device)
static std::mutex boys_mu;
static const double *boys_dev[64] = {nullptr};
static cudaError_t get_boys(const double **out)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lk(boys_mu);
    if (!boys_dev[dev]) {
        void *p = nullptr;
        size_t bytes = sizeof(double) * RCG_BOYS_NROW * RCG_BOYS_NCOL;
        if ((e = cudaMalloc(&p, bytes)) != cudaSuccess) return e;
        if ((e = cudaMemcpy(p, rcg_boys_table_host, bytes, cudaMemcpyHostToDevice)) != cudaSuccess) return e;
        boys_dev[dev] = (const double *)p;
    }
    *out = boys_dev[dev];
    return cudaSuccess;
}

// the handle's device must be the current one: the blob, the Boys grid and the class tables belong to it
static bool on_device(const rcg_basis *b)
{
    int dev = -1;
    return cudaGetDevice(&dev) == cudaSuccess && dev == b->device;
}

// ---------------------------------------------------------------- retained memory pool (one per device)
// Stream-ordered pool for the library's own short-lived device memory: the staging of rcg_eri_batch_host and the
// statistics words of the auto launchers.  It retains its memory between calls (a 500 MB cudaMalloc + cudaFree per call
// cost about a millisecond) and is released at process exit.
static std::mutex pool_mu;
static cudaMemPool_t pools[64] = {};
static bool pool_ok[64] = {};
static cudaError_t get_pool(cudaMemPool_t *out)
{
    int device = 0;
    cudaError_t e = cudaGetDevice(&device);
    if (e != cudaSuccess) return e;
    if (device < 0 || device >= 64) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lk(pool_mu);
    if (!pool_ok[device]) {
        cudaMemPoolProps props = {};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = device;
        if ((e = cudaMemPoolCreate(&pools[device], &props)) != cudaSuccess) return e;
        unsigned long long keep = ~0ull;
        if ((e = cudaMemPoolSetAttribute(pools[device], cudaMemPoolAttrReleaseThreshold, &keep)) != cudaSuccess) return e;
        pool_ok[device] = true;
    }
    *out = pools[device];
    return cudaSuccess;
}

cudaError_t rcg_pool_alloc(void **p, size_t bytes, cudaStream_t stream)
{
    cudaMemPool_t pool;
    cudaError_t e = get_pool(&pool);
    return e != cudaSuccess ? e : cudaMallocFromPoolAsync(p, bytes, pool, stream);
}

// ---------------------------------------------------------------- handle
extern "C" rcg_status rcg_basis_create(rcg_basis **out, int nshell, int nprim, const int32_t *shell_l,
                                       const int32_t *shell_prim_offset, const double *exps,
                                       const double *coefs, const double *centers, void *stream)
{
    if (!out || nshell <= 0 || nprim <= 0 || !shell_l || !shell_prim_offset || !exps || !coefs || !centers)
        return RCG_ERR_INVALID_ARG;
    if (shell_prim_offset[0] != 0 || shell_prim_offset[nshell] != nprim) return RCG_ERR_INVALID_ARG;
    for (int s = 0; s < nshell; ++s) {
        if (shell_l[s] < 0 || shell_l[s] > RCG_LMAX) return RCG_ERR_INVALID_ARG;
        if (shell_prim_offset[s + 1] <= shell_prim_offset[s]) return RCG_ERR_INVALID_ARG;
        if (shell_prim_offset[s + 1] - shell_prim_offset[s] > RCG_KMAX) return RCG_ERR_INVALID_ARG;
    }
    for (int p = 0; p < nprim; ++p)
        if (!(exps[p] > 0.0)) return RCG_ERR_INVALID_ARG;
    rcg_basis *b = new (std::nothrow) rcg_basis;
    if (!b) return RCG_ERR_INVALID_ARG;
    for (int l = 0; l <= RCG_LMAX; ++l) { b->kmin[l] = 1; b->kmax[l] = 1; }
    {
        bool seen[RCG_LMAX + 1] = {false};
        for (int s = 0; s < nshell; ++s) {
            const int l = shell_l[s], k = shell_prim_offset[s + 1] - shell_prim_offset[s];
            if (!seen[l]) { b->kmin[l] = b->kmax[l] = k; seen[l] = true; }
            if (k < b->kmin[l]) b->kmin[l] = k;
            if (k > b->kmax[l]) b->kmax[l] = k;
        }
    }
    cudaError_t e = cudaGetDevice(&b->device);
    if (e != cudaSuccess) { delete b; return cuda_fail(e); }
    // layout of the blob: centers | exps | coefs | prim_off | shell_l   (doubles first: alignment)
    size_t o_cen = 0, o_exp = o_cen + sizeof(double) * 3 * nshell, o_cof = o_exp + sizeof(double) * nprim;
    size_t o_off = o_cof + sizeof(double) * nprim, o_l = o_off + sizeof(int32_t) * (nshell + 1);
    size_t bytes = o_l + sizeof(int32_t) * nshell;
    std::vector<char> host(bytes);
    memcpy(host.data() + o_cen, centers, sizeof(double) * 3 * nshell);
    memcpy(host.data() + o_exp, exps, sizeof(double) * nprim);
    memcpy(host.data() + o_cof, coefs, sizeof(double) * nprim);
    memcpy(host.data() + o_off, shell_prim_offset, sizeof(int32_t) * (nshell + 1));
    memcpy(host.data() + o_l, shell_l, sizeof(int32_t) * nshell);
    if ((e = cudaMalloc(&b->blob, bytes)) != cudaSuccess) { delete b; return cuda_fail(e); }
    cudaStream_t st = (cudaStream_t)stream;
    e = cudaMemcpyAsync(b->blob, host.data(), bytes, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);   // `host` dies at return
    if (e != cudaSuccess) { cudaFree(b->blob); delete b; return cuda_fail(e); }
    char *d = (char *)b->blob;
    b->dev.centers = (const double *)(d + o_cen);
    b->dev.exps = (const double *)(d + o_exp);
    b->dev.coefs = (const double *)(d + o_cof);
    b->dev.prim_off = (const int32_t *)(d + o_off);
    b->dev.shell_l = (const int32_t *)(d + o_l);
    b->dev.nshell = nshell;
    if ((e = get_boys(&b->dev.boys)) != cudaSuccess) { cudaFree(b->blob); delete b; return cuda_fail(e); }
    *out = b;
    return RCG_OK;
}

extern "C" rcg_status rcg_basis_destroy(rcg_basis *b)
{
    if (!b) return RCG_ERR_INVALID_ARG;
    cudaError_t e = cudaFree(b->blob);
    delete b;
    return e == cudaSuccess ? RCG_OK : cuda_fail(e);
}

// ---------------------------------------------------------------- class lookup
// Canonical order: la>=lb, lc>=ld, (la,lb)>=(lc,ld), reached by (ab|cd)=(ba|cd)=(ab|dc)=(cd|ab).
// perm[k] = caller position that supplies canonical position k.
static const RcgClassDesc *find_class(int la, int lb, int lc, int ld, int perm[4])
{
    int l[4] = {la, lb, lc, ld};
    int p[4] = {0, 1, 2, 3};
    for (int k = 0; k < 4; ++k)
        if (l[k] < 0 || l[k] > RCG_LMAX) return nullptr;
    if (l[p[0]] < l[p[1]]) { int t = p[0]; p[0] = p[1]; p[1] = t; }
    if (l[p[2]] < l[p[3]]) { int t = p[2]; p[2] = p[3]; p[3] = t; }
    if (l[p[0]] < l[p[2]] || (l[p[0]] == l[p[2]] && l[p[1]] < l[p[3]])) {
        int t0 = p[0], t1 = p[1];
        p[0] = p[2]; p[1] = p[3]; p[2] = t0; p[3] = t1;
    }
    for (int i = 0; i < rcg_class_count; ++i) {
        const RcgClassDesc *d = rcg_class_table[i];
        if (d->l[0] == l[p[0]] && d->l[1] == l[p[1]] && d->l[2] == l[p[2]] && d->l[3] == l[p[3]]) {
            for (int k = 0; k < 4; ++k) perm[k] = p[k];
            return d;
        }
    }
    return nullptr;
}

static bool use_global(const RcgClassDesc *d, int tier) { return tier == RCG_TIER_GLOBAL || d->launch == nullptr; }

// scratch of one launch: the slot buffer of the global tier, or H + the half-transformed block of one chunk of the heavy
// block tier (csrc/rcg_sides.h), else nothing
static size_t class_workspace_bytes(const RcgClassDesc *d, int tier, int64_t n)
{
    if (n <= 0) return 0;
    if (use_global(d, tier)) return rcg_global_workspace_bytes(*d, n);
    if (d->ws_quartet_doubles > 0) return sizeof(double) * (size_t)d->ws_quartet_doubles * (size_t)rcg_heavy_chunk(d->ws_quartet_doubles, n);
    return 0;
}

extern "C" rcg_status rcg_eri_workspace_bytes_tier(const rcg_basis *b, int tier, int la, int lb, int lc, int ld,
                                                   int64_t nquartet, size_t *bytes)
{
    if (!b || !bytes || nquartet < 0 || !on_device(b)) return RCG_ERR_INVALID_ARG;
    int perm[4];
    const RcgClassDesc *d = find_class(la, lb, lc, ld, perm);
    if (!d) return (la < 0 || lb < 0 || lc < 0 || ld < 0 || la > RCG_LMAX || lb > RCG_LMAX || lc > RCG_LMAX || ld > RCG_LMAX)
                       ? RCG_ERR_INVALID_ARG : RCG_ERR_UNSUPPORTED_CLASS;
    if (tier != 0 && tier != RCG_TIER_GLOBAL && tier != d->tier && !(d->tier == RCG_TIER_REGISTER && tier == RCG_TIER_WARP))
        return RCG_ERR_UNSUPPORTED_CLASS;
    *bytes = class_workspace_bytes(d, tier, nquartet);
    return RCG_OK;
}

extern "C" rcg_status rcg_eri_workspace_bytes(const rcg_basis *b, int la, int lb, int lc, int ld,
                                              int64_t nquartet, size_t *bytes)
{
    return rcg_eri_workspace_bytes_tier(b, 0, la, lb, lc, ld, nquartet, bytes);
}

static rcg_status eri_batch_impl(const rcg_basis *b, int tier, int uniform, int la, int lb, int lc, int ld,
                                 const int32_t *quartets, int64_t nquartet, double *out,
                                 void *workspace, size_t workspace_bytes, void *stream)
{
    if (!b || nquartet < 0 || !on_device(b)) return RCG_ERR_INVALID_ARG;
    int perm[4];
    const RcgClassDesc *d = find_class(la, lb, lc, ld, perm);
    if (!d) return (la < 0 || lb < 0 || lc < 0 || ld < 0 || la > RCG_LMAX || lb > RCG_LMAX || lc > RCG_LMAX || ld > RCG_LMAX)
                       ? RCG_ERR_INVALID_ARG : RCG_ERR_UNSUPPORTED_CLASS;
    if (tier != 0 && tier != RCG_TIER_GLOBAL && tier != d->tier && !(d->tier == RCG_TIER_REGISTER && tier == RCG_TIER_WARP))
        return RCG_ERR_UNSUPPORTED_CLASS;
    if (nquartet == 0) return RCG_OK;
    if (!quartets || !out || ((uintptr_t)quartets & 15) != 0) return RCG_ERR_INVALID_ARG;
    const bool glob = use_global(d, tier);
    size_t need = class_workspace_bytes(d, tier, nquartet);
    if (need > 0 && (!workspace || workspace_bytes < need)) return RCG_ERR_WORKSPACE_TOO_SMALL;
    RcgLaunch a;
    a.basis = b->dev;
    a.quartets = quartets;
    a.n = nquartet;
    a.out = out;
    a.workspace = (double *)workspace;
    a.stream = (cudaStream_t)stream;
    a.stat = nullptr;
    a.stat_reg = nullptr;
    a.force_tier = tier;
    a.uniform_k4 = uniform;
    a.bf_off = nullptr; a.D = nullptr; a.Jt = nullptr; a.Kt = nullptr; a.nbf = 0;
    RcgStatHolder holder = {a.stream, nullptr};
    a.stat_holder = &holder;
    for (int l = 0; l <= RCG_LMAX; ++l) { a.kmin[l] = b->kmin[l]; a.kmax[l] = b->kmax[l]; }
    const int lcall[4] = {la, lb, lc, ld};
    int64_t cstride[4];   // caller strides: d fastest
    cstride[3] = 1;
    cstride[2] = 2 * ld + 1;
    cstride[1] = cstride[2] * (2 * lc + 1);
    cstride[0] = cstride[1] * (2 * lb + 1);
    a.out_stride = cstride[0] * (2 * la + 1);
    for (int k = 0; k < 4; ++k) {
        a.perm[k] = perm[k];
        a.nsph[k] = 2 * lcall[perm[k]] + 1;
        a.lcan[k] = lcall[perm[k]];
        a.ostride[k] = cstride[perm[k]];
    }
    cudaError_t e = glob ? rcg_global_launch(*d, a) : d->launch(a);
    const cudaError_t e2 = rcg_stat_release(holder);       // stream-ordered, after the kernels enqueued above
    if (e == cudaSuccess) e = e2;
    return e == cudaSuccess ? RCG_OK : cuda_fail(e);
}

extern "C" rcg_status rcg_eri_batch_tier(const rcg_basis *b, int tier, int la, int lb, int lc, int ld,
                                         const int32_t *quartets, int64_t nquartet, double *out,
                                         void *workspace, size_t workspace_bytes, void *stream)
{
    return eri_batch_impl(b, tier, 0, la, lb, lc, ld, quartets, nquartet, out, workspace, workspace_bytes, stream);
}

extern "C" rcg_status rcg_eri_batch(const rcg_basis *b, int la, int lb, int lc, int ld, const int32_t *quartets,
                                    int64_t nquartet, double *out, void *workspace, size_t workspace_bytes,
                                    void *stream)
{
    return eri_batch_impl(b, 0, 0, la, lb, lc, ld, quartets, nquartet, out, workspace, workspace_bytes, stream);
}

extern "C" rcg_status rcg_eri_batch_uniform(const rcg_basis *b, int la, int lb, int lc, int ld, const int32_t *quartets,
                                            int64_t nquartet, double *out, void *workspace, size_t workspace_bytes,
                                            void *stream)
{
    return eri_batch_impl(b, 0, 1, la, lb, lc, ld, quartets, nquartet, out, workspace, workspace_bytes, stream);
}

// ---------------------------------------------------------------- first derivatives (csrc/eri_grad.cu)
extern "C" rcg_status rcg_eri_grad_supported(int la, int lb, int lc, int ld, int *supported, size_t *smem_bytes)
{
    if (!supported) return RCG_ERR_INVALID_ARG;
    const int l[4] = {la, lb, lc, ld};
    for (int k = 0; k < 4; ++k)
        if (l[k] < 0 || l[k] > RCG_LMAX) return RCG_ERR_INVALID_ARG;
    *supported = rcg_grad_supported(l, smem_bytes) ? 1 : 0;
    return RCG_OK;
}

static rcg_status grad_batch_impl(const rcg_basis *b, int la, int lb, int lc, int ld, const int32_t *quartets,
                                  int64_t nquartet, long long k4hint, double *out, void *stream)
{
    if (!b || nquartet < 0 || !on_device(b)) return RCG_ERR_INVALID_ARG;
    RcgGradLaunch a;
    a.l[0] = la; a.l[1] = lb; a.l[2] = lc; a.l[3] = ld;
    for (int k = 0; k < 4; ++k)
        if (a.l[k] < 0 || a.l[k] > RCG_LMAX) return RCG_ERR_INVALID_ARG;
    if (!rcg_grad_supported(a.l, nullptr)) return RCG_ERR_UNSUPPORTED_CLASS;
    if (nquartet == 0) return RCG_OK;
    if (!quartets || !out || ((uintptr_t)quartets & 15) != 0) return RCG_ERR_INVALID_ARG;
    a.basis = b->dev;
    a.quartets = quartets;
    a.n = nquartet;
    a.out = out;
    a.stream = (cudaStream_t)stream;
    a.k4max = 1;
    for (int k = 0; k < 4; ++k) a.k4max *= b->kmax[a.l[k]];
    a.k4_promised = k4hint > 0;
    if (k4hint > 0) a.k4max = k4hint;
    const cudaError_t e = rcg_grad_launch(a);
    return e == cudaSuccess ? RCG_OK : cuda_fail(e);
}

extern "C" rcg_status rcg_eri_grad_batch(const rcg_basis *b, int la, int lb, int lc, int ld, const int32_t *quartets,
                                         int64_t nquartet, double *out, void *stream)
{
    return grad_batch_impl(b, la, lb, lc, ld, quartets, nquartet, 0, out, stream);
}

extern "C" rcg_status rcg_eri_grad_batch_uniform(const rcg_basis *b, int la, int lb, int lc, int ld, const int32_t *quartets,
                                                 int64_t nquartet, int64_t k4, double *out, void *stream)
{
    if (k4 <= 0) return RCG_ERR_INVALID_ARG;
    return grad_batch_impl(b, la, lb, lc, ld, quartets, nquartet, k4, out, stream);
}

// ---------------------------------------------------------------- Fock build: integrals digested without a trip through HBM
// Register-tier classes on long lists with one K4: the digestion runs in the class kernel's epilogue.  Everything
// else: the class kernel writes chunks of at most 1 GiB into the workspace and rcg_jk_digest (the paper's buffered form) reads
// them.  (L2-sized chunks of 48 MB measured SLOWER on the cfg5 Fock pass, 7.65 against 7.51 s: the block-tier kernels and the digestion
// lose more to short launches -- a few waves each -- than the L2 residency of the blocks gains.)
#define RCG_FOCK_CHUNK_BYTES (1ull << 30)
#define RCG_FOCK_REG_MIN 8192

static int64_t fock_chunk(size_t nout, int64_t n)
{
    int64_t c = (int64_t)(RCG_FOCK_CHUNK_BYTES / (nout * sizeof(double)));
    if (c < 256) c = 256;
    return n < c ? n : c;
}

// inline digestion: the register-tier kernels (a thread per quartet) want a long list with one K4, the warp-tier kernels take any list
static bool fock_fused(const RcgClassDesc *d, int64_t n, int uniform_k4)
{
    if (!d->launch_fock) return false;
    return d->fock_kind == 1 ? (uniform_k4 && n >= RCG_FOCK_REG_MIN) : true;
}

extern "C" rcg_status rcg_fock_workspace_bytes(const rcg_basis *b, int la, int lb, int lc, int ld, int64_t nquartet,
                                               int uniform_k4, size_t *bytes)
{
    if (!b || !bytes || nquartet < 0 || !on_device(b)) return RCG_ERR_INVALID_ARG;
    int perm[4];
    const RcgClassDesc *d = find_class(la, lb, lc, ld, perm);
    if (!d) return RCG_ERR_UNSUPPORTED_CLASS;
    if (perm[0] != 0 || perm[1] != 1 || perm[2] != 2 || perm[3] != 3) return RCG_ERR_INVALID_ARG;
    *bytes = 0;
    if (nquartet == 0 || fock_fused(d, nquartet, uniform_k4)) return RCG_OK;
    const size_t nout = (size_t)(2 * la + 1) * (2 * lb + 1) * (2 * lc + 1) * (2 * ld + 1);
    const int64_t chunk = fock_chunk(nout, nquartet);
    *bytes = ((sizeof(double) * nout * (size_t)chunk + 255) & ~(size_t)255) + class_workspace_bytes(d, 0, chunk);
    return RCG_OK;
}

extern "C" rcg_status rcg_fock_batch(const rcg_basis *b, int la, int lb, int lc, int ld, const int32_t *quartets,
                                     int64_t nquartet, int uniform_k4, const int32_t *shell_bf_offset, const double *D,
                                     double *Jt, double *Kt, int nbf, void *workspace, size_t workspace_bytes, void *stream)
{
    if (!b || nquartet < 0 || nbf <= 0 || !on_device(b)) return RCG_ERR_INVALID_ARG;
    int perm[4];
    const RcgClassDesc *d = find_class(la, lb, lc, ld, perm);
    if (!d) return (la < 0 || lb < 0 || lc < 0 || ld < 0 || la > RCG_LMAX || lb > RCG_LMAX || lc > RCG_LMAX || ld > RCG_LMAX)
                       ? RCG_ERR_INVALID_ARG : RCG_ERR_UNSUPPORTED_CLASS;
    if (perm[0] != 0 || perm[1] != 1 || perm[2] != 2 || perm[3] != 3) return RCG_ERR_INVALID_ARG;      // canonical class order only
    if (nquartet == 0) return RCG_OK;
    if (!quartets || !shell_bf_offset || !D || !Jt || !Kt || ((uintptr_t)quartets & 15) != 0) return RCG_ERR_INVALID_ARG;
    if (fock_fused(d, nquartet, uniform_k4)) {
        RcgLaunch a = {};
        a.basis = b->dev; a.quartets = quartets; a.n = nquartet; a.stream = (cudaStream_t)stream;
        a.uniform_k4 = uniform_k4;
        for (int l = 0; l <= RCG_LMAX; ++l) { a.kmin[l] = b->kmin[l]; a.kmax[l] = b->kmax[l]; }
        const int lcall[4] = {la, lb, lc, ld};
        for (int k = 0; k < 4; ++k) { a.perm[k] = k; a.nsph[k] = 2 * lcall[k] + 1; a.lcan[k] = lcall[k]; }
        a.bf_off = shell_bf_offset; a.D = D; a.Jt = Jt; a.Kt = Kt; a.nbf = nbf;
        const cudaError_t e = d->launch_fock(a);
        return e == cudaSuccess ? RCG_OK : cuda_fail(e);
    }
    size_t need = 0;
    rcg_status s = rcg_fock_workspace_bytes(b, la, lb, lc, ld, nquartet, uniform_k4, &need);
    if (s != RCG_OK) return s;
    if (!workspace || workspace_bytes < need) return RCG_ERR_WORKSPACE_TOO_SMALL;
    const size_t nout = (size_t)(2 * la + 1) * (2 * lb + 1) * (2 * lc + 1) * (2 * ld + 1);
    const int64_t chunk = fock_chunk(nout, nquartet);
    const size_t blk_bytes = (sizeof(double) * nout * (size_t)chunk + 255) & ~(size_t)255;
    double *blocks = (double *)workspace;
    void *cws = (char *)workspace + blk_bytes;
    for (int64_t off = 0; off < nquartet; off += chunk) {
        const int64_t cn = nquartet - off < chunk ? nquartet - off : chunk;
        s = eri_batch_impl(b, 0, uniform_k4, la, lb, lc, ld, quartets + 4 * off, cn, blocks, cws, workspace_bytes - blk_bytes, stream);
        if (s != RCG_OK) return s;
        s = rcg_jk_digest(la, lb, lc, ld, quartets + 4 * off, cn, blocks, shell_bf_offset, D, Jt, Kt, nbf, stream);
        if (s != RCG_OK) return s;
    }
    return RCG_OK;
}

// HOST list and HOST output.  The batch is cut into chunks of at least 32 MB of output (never below 8,192 quartets,
// which is also what the register tier wants for the classes that have one); the kernel of chunk k + 1 runs
// while chunk k is copied back on a second stream, so with pinned host memory the call takes about the time of the
// device-to-host copy alone ((dd|dd), 100,000 quartets: 500 MB).  Pageable memory works, without the overlap.
extern "C" rcg_status rcg_eri_batch_host(const rcg_basis *b, int la, int lb, int lc, int ld,
                                         const int32_t *quartets_host, int64_t nquartet, double *out_host,
                                         void *stream)
{
    if (!b || nquartet < 0 || !on_device(b)) return RCG_ERR_INVALID_ARG;
    if (nquartet == 0) return RCG_OK;
    if (!quartets_host || !out_host) return RCG_ERR_INVALID_ARG;
    rcg_status s = rcg_class_info(la, lb, lc, ld, nullptr, nullptr, nullptr);
    if (s != RCG_OK) return s;
    const size_t nout = (size_t)(2 * la + 1) * (2 * lb + 1) * (2 * lc + 1) * (2 * ld + 1);
    int64_t chunk = (int64_t)((32u << 20) / (nout * sizeof(double))) + 1;
    if (chunk < 8192) chunk = 8192;
    if (chunk > nquartet) chunk = nquartet;
    size_t wsb = 0;
    if ((s = rcg_eri_workspace_bytes(b, la, lb, lc, ld, chunk, &wsb)) != RCG_OK) return s;
    // the copy stream and the two events are PER CALL: concurrent callers on one device must not re-record each other's events
    cudaMemPool_t pool;
    cudaError_t e = get_pool(&pool);
    if (e != cudaSuccess) return cuda_fail(e);
    cudaStream_t copy = nullptr;
    cudaEvent_t ev_k = nullptr, ev_c = nullptr;
    if ((e = cudaStreamCreateWithFlags(&copy, cudaStreamNonBlocking)) != cudaSuccess) return cuda_fail(e);
    if ((e = cudaEventCreateWithFlags(&ev_k, cudaEventDisableTiming)) != cudaSuccess) { cudaStreamDestroy(copy); return cuda_fail(e); }
    if ((e = cudaEventCreateWithFlags(&ev_c, cudaEventDisableTiming)) != cudaSuccess) { cudaEventDestroy(ev_k); cudaStreamDestroy(copy); return cuda_fail(e); }
    cudaStream_t st = (cudaStream_t)stream;
    const size_t qb = sizeof(int32_t) * 4 * (size_t)nquartet, ob = sizeof(double) * (size_t)nquartet * nout;
    void *dq = nullptr, *dout = nullptr, *dws = nullptr;
    e = cudaMallocFromPoolAsync(&dq, qb, pool, st);
    if (e == cudaSuccess) e = cudaMallocFromPoolAsync(&dout, ob, pool, st);
    if (e == cudaSuccess && wsb) e = cudaMallocFromPoolAsync(&dws, wsb, pool, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(dq, quartets_host, qb, cudaMemcpyHostToDevice, st);
    for (int64_t off = 0; e == cudaSuccess && s == RCG_OK && off < nquartet; off += chunk) {
        const int64_t cn = nquartet - off < chunk ? nquartet - off : chunk;
        s = rcg_eri_batch(b, la, lb, lc, ld, (const int32_t *)dq + 4 * off, cn, (double *)dout + off * nout, dws, wsb, stream);
        if (s != RCG_OK) break;
        e = cudaEventRecord(ev_k, st);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(copy, ev_k, 0);
        if (e == cudaSuccess) e = cudaMemcpyAsync(out_host + off * nout, (double *)dout + off * nout, sizeof(double) * cn * nout,
                                                  cudaMemcpyDeviceToHost, copy);
    }
    // the caller's stream continues after the last copy; then the staging goes back to the pool
    cudaError_t e2 = cudaEventRecord(ev_c, copy);
    if (e2 == cudaSuccess) e2 = cudaStreamWaitEvent(st, ev_c, 0);
    if (dq) cudaFreeAsync(dq, st);
    if (dout) cudaFreeAsync(dout, st);
    if (dws) cudaFreeAsync(dws, st);
    cudaError_t e3 = cudaStreamSynchronize(st);
    cudaEventDestroy(ev_k);
    cudaEventDestroy(ev_c);
    cudaStreamDestroy(copy);
    if (e == cudaSuccess) e = e2;
    if (e == cudaSuccess) e = e3;
    if (e != cudaSuccess) return cuda_fail(e);
    return s;
}

// ---------------------------------------------------------------- validation
__global__ void rcg_validate_kernel(RcgBasisDev b, const int32_t *q, int64_t n, int l0, int l1, int l2, int l3,
                                    int *bad)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int l[4] = {l0, l1, l2, l3};
    for (int k = 0; k < 4; ++k) {
        int s = q[4 * i + k];
        if (s < 0 || s >= b.nshell || b.shell_l[s] != l[k]) { atomicExch(bad, 1); return; }
    }
}

extern "C" rcg_status rcg_validate_batch(const rcg_basis *b, int la, int lb, int lc, int ld, const int32_t *quartets,
                                         int64_t nquartet, void *stream)
{
    if (!b || nquartet < 0 || (nquartet > 0 && !quartets) || !on_device(b)) return RCG_ERR_INVALID_ARG;
    if (nquartet == 0) return RCG_OK;
    int *bad = nullptr, h = 0;
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e = cudaMalloc((void **)&bad, sizeof(int));
    if (e != cudaSuccess) return cuda_fail(e);
    e = cudaMemsetAsync(bad, 0, sizeof(int), st);
    if (e == cudaSuccess) {
        rcg_validate_kernel<<<(unsigned)((nquartet + 255) / 256), 256, 0, st>>>(b->dev, quartets, nquartet, la, lb, lc, ld, bad);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(&h, bad, sizeof(int), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(bad);
    if (e != cudaSuccess) return cuda_fail(e);
    return h ? RCG_ERR_CLASS_MISMATCH : RCG_OK;
}

// ---------------------------------------------------------------- Boys alone
__global__ void rcg_boys_kernel(int mmax, const double *T, int64_t n, double *out, const double *tab)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double F[17];
    rcg_boys<-1>(mmax, T[i], 1.0, tab, F);
    for (int m = 0; m <= mmax; ++m) out[i * (mmax + 1) + m] = F[m];
}

extern "C" rcg_status rcg_boys(int mmax, const double *T, int64_t n, double *out, void *stream)
{
    if (mmax < 0 || mmax > 16 || n < 0 || (n > 0 && (!T || !out))) return RCG_ERR_INVALID_ARG;
    if (n == 0) return RCG_OK;
    const double *tab = nullptr;
    cudaError_t e = get_boys(&tab);
    if (e != cudaSuccess) return cuda_fail(e);
    rcg_boys_kernel<<<(unsigned)((n + 127) / 128), 128, 0, (cudaStream_t)stream>>>(mmax, T, n, out, tab);
    e = cudaGetLastError();
    return e == cudaSuccess ? RCG_OK : cuda_fail(e);
}

// ---------------------------------------------------------------- static facts
extern "C" rcg_status rcg_class_info(int la, int lb, int lc, int ld, int *tier, int64_t *flops_per_prim_quartet,
                                     int64_t *flops_per_quartet)
{
    int perm[4];
    const RcgClassDesc *d = find_class(la, lb, lc, ld, perm);
    if (!d) return RCG_ERR_UNSUPPORTED_CLASS;
    if (tier) *tier = d->launch ? d->tier : RCG_TIER_GLOBAL;
    if (flops_per_prim_quartet) *flops_per_prim_quartet = d->flops_prim;
    if (flops_per_quartet) *flops_per_quartet = d->flops_quartet;
    return RCG_OK;
}

extern "C" int rcg_num_classes(void) { return rcg_class_count; }

extern "C" rcg_status rcg_class_at(int i, int *la, int *lb, int *lc, int *ld)
{
    if (i < 0 || i >= rcg_class_count) return RCG_ERR_INVALID_ARG;
    const RcgClassDesc *d = rcg_class_table[i];
    if (la) *la = d->l[0];
    if (lb) *lb = d->l[1];
    if (lc) *lc = d->l[2];
    if (ld) *ld = d->l[3];
    return RCG_OK;
}

extern "C" const char *rcg_status_string(rcg_status s)
{
    switch (s) {
    case RCG_OK: return "ok";
    case RCG_ERR_INVALID_ARG: return "invalid argument";
    case RCG_ERR_UNSUPPORTED_CLASS: return "unsupported angular class";
    case RCG_ERR_WORKSPACE_TOO_SMALL: return "workspace too small";
    case RCG_ERR_CUDA: return "CUDA error";
    case RCG_ERR_CLASS_MISMATCH: return "quartet list does not match the angular class";
    case RCG_ERR_STATIC_SCRATCH_LIMIT: return "batch exceeds the static scratch of rcg_eri_batch_static (RCG_STATIC_SCRATCH_BYTES = 32 MiB; see rcg_eri_batch_static_max_quartets)";
    default: return "unknown status";
    }
}

extern "C" int rcg_last_cuda_error(void) { return tl_cuda_error; }
