// tier_global.cu -- RCG_TIER_GLOBAL: table-driven kernel, one thread per shell quartet, every
// intermediate in an interleaved global scratch (slot-major, thread-minor: slot s of thread t is
// ws[s * nthreads + t], so the 32 lanes of a warp touch one 256-byte segment per access) -- the
// layout PAPER.md:263-265 gives for the paper's Tier 2.  Works for every generated class; it is
// the only tier for the heaviest ones ((ff|..), (gg|gg)) and the cross-check for the others.
// Steps per quartet follow Alg. 2: H <- 0; for each primitive quartet
// {pair quantities, Boys, VRR in family order, H += V}; bra HRR + Ta,Tb per ket column;
// ket HRR + Tc,Td per bra row; store.
#include <mutex>
#include <map>
#include "rcg_device.cuh"

struct GDev {                 // device copies of one class's tables
    const uint32_t *vrr_fam; const int32_t *tslots;
    const uint32_t *bra_ops; const uint32_t *ket_ops;
    const uint16_t *bra_out; const uint16_t *ket_out;
    const double *consts;
    int n_fam, n_targets, nA, nC, n_vslots;
    int n_bra_ops, bra_nin, bra_nslots, bra_nout;
    int n_ket_ops, ket_nin, ket_nslots, ket_nout;
    int L;
};

__device__ __forceinline__ void run_lin(const uint32_t *__restrict__ ops, int nops, const double *__restrict__ consts,
                                        double *loc, int64_t T, double X0, double X1, double X2)
{
    for (int i = 0; i < nops; ++i) {
        const uint32_t w0 = __ldg(ops + 2 * i), w1 = __ldg(ops + 2 * i + 1);
        const int dst = w0 >> 16, src = w0 & 0xffff, sel = w1 & 0xffff;
        const double s = loc[(int64_t)src * T];
        double c;
        if (sel == 0) c = 1.0;
        else if (sel == 1) c = X0;
        else if (sel == 2) c = X1;
        else if (sel == 3) c = X2;
        else c = __ldg(consts + (sel - 4));
        if (w1 >> 16) loc[(int64_t)dst * T] = c * s;
        else loc[(int64_t)dst * T] = fma(c, s, loc[(int64_t)dst * T]);
    }
}

__global__ void __launch_bounds__(128) rcg_eri_global_kernel(GDev g, RcgLaunch a)
{
    const int64_t T = (int64_t)gridDim.x * blockDim.x;
    const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    double *V = a.workspace + tid;                               // VRR slots
    double *H = V + (int64_t)g.n_vslots * T;                      // [nA][nC] contracted targets
    double *Bh = H + (int64_t)g.n_targets * T;                    // [bra_nout][nC] half-transformed
    double *loc = Bh + (int64_t)g.bra_nout * g.nC * T;            // Phase-2 private slots
    const RcgBasisDev &b = a.basis;
    for (int64_t q = tid; q < a.n; q += T) {
        int sh[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) sh[k] = a.quartets[4 * q + a.perm[k]];
        double R[4][3];
#pragma unroll
        for (int k = 0; k < 4; ++k)
#pragma unroll
            for (int t = 0; t < 3; ++t) R[k][t] = b.centers[3 * sh[k] + t];
        for (int t = 0; t < g.n_targets; ++t) H[(int64_t)t * T] = 0.0;
        const int p0 = b.prim_off[sh[0]], p0e = b.prim_off[sh[0] + 1];
        const int p1 = b.prim_off[sh[1]], p1e = b.prim_off[sh[1] + 1];
        const int p2 = b.prim_off[sh[2]], p2e = b.prim_off[sh[2] + 1];
        const int p3 = b.prim_off[sh[3]], p3e = b.prim_off[sh[3] + 1];
        for (int i = p0; i < p0e; ++i)
        for (int j = p1; j < p1e; ++j)
        for (int k = p2; k < p2e; ++k)
        for (int l = p3; l < p3e; ++l) {
            RcgPrim p;
            rcg_prim_setup(p, R[0], R[1], R[2], R[3], b.exps[i], b.exps[j], b.exps[k], b.exps[l],
                           b.coefs[i] * b.coefs[j] * b.coefs[k] * b.coefs[l]);
            double F[17];
            rcg_boys<-1>(g.L, p.T, p.pref, b.boys, F);
            for (int m = 0; m <= g.L; ++m) V[(int64_t)m * T] = F[m];
            for (int f = 0; f < g.n_fam; ++f) {
                const uint32_t *w = g.vrr_fam + 5 * f;
                const int64_t od = __ldg(w), o1 = __ldg(w + 1), o3 = __ldg(w + 2), o5 = __ldg(w + 3);
                const uint32_t meta = __ldg(w + 4);
                const int mlo = meta & 31, nm = (meta >> 5) & 31, ket = (meta >> 10) & 1, ax = (meta >> 11) & 3;
                const int n2 = (meta >> 13) & 15, nx = (meta >> 17) & 15;
                const double c1 = ket ? p.QC[ax] : p.PA[ax];
                const double c2 = ket ? p.WQ[ax] : p.WP[ax];
                const double k3 = (double)n2 * (ket ? p.he : p.hz);
                const double r3 = ket ? p.re : p.rz;
                const double k5 = (double)nx * p.hze;
                for (int m = mlo; m < mlo + nm; ++m) {
                    double v = c1 * V[(o1 + m) * T];
                    v = fma(c2, V[(o1 + m + 1) * T], v);
                    if (n2) v = fma(k3, fma(-r3, V[(o3 + m + 1) * T], V[(o3 + m) * T]), v);
                    if (nx) v = fma(k5, V[(o5 + m + 1) * T], v);
                    V[(od + m) * T] = v;
                }
            }
            for (int t = 0; t < g.n_targets; ++t) H[(int64_t)t * T] += V[(int64_t)__ldg(g.tslots + t) * T];
        }
        // Phase 2, bra side: for every ket column c
        const double AB0 = R[0][0] - R[1][0], AB1 = R[0][1] - R[1][1], AB2 = R[0][2] - R[1][2];
        const double CD0 = R[2][0] - R[3][0], CD1 = R[2][1] - R[3][1], CD2 = R[2][2] - R[3][2];
        for (int c = 0; c < g.nC; ++c) {
            for (int k = 0; k < g.nA; ++k) loc[(int64_t)k * T] = H[(int64_t)(k * g.nC + c) * T];
            run_lin(g.bra_ops, g.n_bra_ops, g.consts, loc, T, AB0, AB1, AB2);
            for (int o = 0; o < g.bra_nout; ++o) Bh[(int64_t)(o * g.nC + c) * T] = loc[(int64_t)__ldg(g.bra_out + o) * T];
        }
        // ket side: for every (spherical) bra row o = ia*nsph(lb)+ib
        double *out = a.out + q * a.out_stride;
        const int nsb = a.nsph[1], nsd = a.nsph[3];
        for (int o = 0; o < g.bra_nout; ++o) {
            for (int k = 0; k < g.nC; ++k) loc[(int64_t)k * T] = Bh[(int64_t)(o * g.nC + k) * T];
            run_lin(g.ket_ops, g.n_ket_ops, g.consts, loc, T, CD0, CD1, CD2);
            const int64_t obase = (int64_t)(o / nsb) * a.ostride[0] + (int64_t)(o % nsb) * a.ostride[1];
            for (int r = 0; r < g.ket_nout; ++r)
                out[obase + (int64_t)(r / nsd) * a.ostride[2] + (int64_t)(r % nsd) * a.ostride[3]] =
                    loc[(int64_t)__ldg(g.ket_out + r) * T];
        }
    }
}

// ---------------------------------------------------------------- host side
static size_t slots_per_thread(const RcgGlobalTables &t)
{
    int p2 = t.bra_nslots > t.ket_nslots ? t.bra_nslots : t.ket_nslots;
    return (size_t)t.n_vslots + (size_t)t.n_targets + (size_t)t.bra_nout * t.nC + (size_t)p2;
}

// threads of one launch: whole blocks of 128, at most 8 blocks per SM, and at most 6 GiB of scratch
static int64_t global_threads(const RcgClassDesc &d, int64_t n)
{
    int dev = 0, nsm = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    int64_t t = ((n + 127) / 128) * 128;
    int64_t cap = (int64_t)nsm * 8 * 128;
    int64_t memcap = (int64_t)((6ull << 30) / (slots_per_thread(d.g) * 8)) / 128 * 128;
    if (memcap < 128) memcap = 128;
    if (t > cap) t = cap;
    if (t > memcap) t = memcap;
    return t;
}

size_t rcg_global_workspace_bytes(const RcgClassDesc &d, int64_t n)
{
    if (n <= 0) return 0;
    return slots_per_thread(d.g) * 8 * (size_t)global_threads(d, n);
}

static std::mutex g_mu;
static std::map<std::pair<int, const RcgClassDesc *>, GDev> g_cache;

template <class T>
static cudaError_t upload(const T *h, size_t n, const T **d)
{
    void *p = nullptr;
    cudaError_t e = cudaMalloc(&p, (n ? n : 1) * sizeof(T));
    if (e != cudaSuccess) return e;
    e = cudaMemcpy(p, h, n * sizeof(T), cudaMemcpyHostToDevice);
    *d = (const T *)p;
    return e;
}

static cudaError_t get_tables(const RcgClassDesc &d, GDev *out)
{
    int dev = 0;
    cudaGetDevice(&dev);
    std::lock_guard<std::mutex> lk(g_mu);
    auto key = std::make_pair(dev, &d);
    auto it = g_cache.find(key);
    if (it != g_cache.end()) { *out = it->second; return cudaSuccess; }
    const RcgGlobalTables &t = d.g;
    GDev g;
    cudaError_t e;
    if ((e = upload(t.vrr_fam, (size_t)t.n_fam * 5, &g.vrr_fam)) != cudaSuccess) return e;
    if ((e = upload(t.tslots, (size_t)t.n_targets, &g.tslots)) != cudaSuccess) return e;
    if ((e = upload(t.bra_ops, (size_t)t.n_bra_ops * 2, &g.bra_ops)) != cudaSuccess) return e;
    if ((e = upload(t.ket_ops, (size_t)t.n_ket_ops * 2, &g.ket_ops)) != cudaSuccess) return e;
    if ((e = upload(t.bra_out, (size_t)t.bra_nout, &g.bra_out)) != cudaSuccess) return e;
    if ((e = upload(t.ket_out, (size_t)t.ket_nout, &g.ket_out)) != cudaSuccess) return e;
    if ((e = upload(t.consts, (size_t)t.n_consts, &g.consts)) != cudaSuccess) return e;
    g.n_fam = t.n_fam; g.n_targets = t.n_targets; g.nA = t.nA; g.nC = t.nC; g.n_vslots = t.n_vslots;
    g.n_bra_ops = t.n_bra_ops; g.bra_nin = t.bra_nin; g.bra_nslots = t.bra_nslots; g.bra_nout = t.bra_nout;
    g.n_ket_ops = t.n_ket_ops; g.ket_nin = t.ket_nin; g.ket_nslots = t.ket_nslots; g.ket_nout = t.ket_nout;
    g.L = d.l[0] + d.l[1] + d.l[2] + d.l[3];
    g_cache[key] = g;
    *out = g;
    return cudaSuccess;
}

cudaError_t rcg_global_launch(const RcgClassDesc &d, const RcgLaunch &a)
{
    GDev g;
    cudaError_t e = get_tables(d, &g);
    if (e != cudaSuccess) return e;
    int64_t threads = global_threads(d, a.n);
    rcg_eri_global_kernel<<<(unsigned)(threads / 128), 128, 0, a.stream>>>(g, a);
    return cudaGetLastError();
}
