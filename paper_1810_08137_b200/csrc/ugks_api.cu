// ugks_api.cu -- the C ABI of include/ugks.h: context, workspace carving, launch sequencing.
#include "../../include/ugks.h"
#include "ugks_common.cuh"
#include "ugks_jit.h"

#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

struct ugks_ctx {
    UgksParams P;
    KGeom *gm, *gu;           // launch geometries of k_cell_moments / k_flux_update (P.nchunk, P.R, ... mirror gm)
    JitKernel *km, *ku;       // the run-time specialised kernels of these geometries (ugks_jit.cu)
    int device;               // the device the context was created on; every entry point runs there
    cudaStream_t st;
    int cur;                  // which of f[2] / W[2] holds the current state
    int have_state, have_res;
    long steps, launches;
    int resblocks, nchunk_alloc;
    double *res_dev, *bcprim_dev, *Wf_dev;
    double *ghost, *wallg, *Wb, *wallG, *ghostmom;   // non-const aliases of the P fields
    int4 *chunks_dev;
    double *vhost, *uhost, *wvhost, *wuhost;   // host copies of the velocity nodes and weights (chunking, JIT constants)
    size_t cells;
    int profile;              // option "profile": time every kernel of ugks_step with CUDA events
    int poison;               // option "poison": NaN-fill every SM's shared memory before each f-sized kernel (test aid)
    cudaEvent_t *ev; int nev, nev_used;
    double kms[5]; long kcnt[5];
    // CUDA graph of two consecutive steps (launch-bound meshes): captured on an internal stream, replayed between two events
    int graph_mode;           // option "graph": -1 auto (on below 3e7 points per step), 0 off, 1 on
    long graph_launches;      // kernels inside a graph
    cudaStream_t gst; cudaGraphExec_t gexec[2]; cudaEvent_t gin, gout;       // gexec[p]: two steps starting from state parity p
    char err[256];
};

static char g_err[256] = "";
extern "C" { static void drop_graph(ugks_ctx *c); }
static int fail(ugks_ctx *c, int code, const char *fmt, const char *detail)
{
    char *dst = c ? c->err : g_err;
    snprintf(dst, 256, fmt, detail ? detail : "");
    return code;
}
static int cuda_fail(ugks_ctx *c, cudaError_t e, const char *where)
{
    char buf[200];
    snprintf(buf, sizeof buf, "%s: %s", where, cudaGetErrorString(e));
    return fail(c, UGKS_ECUDA, "CUDA error in %s", buf);
}
#define CK(call, where) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(c, e_, where); } while (0)

// every entry point runs on the device the context was created on (function attributes, streams and the workspace live there)
struct DevGuard {
    int prev, changed;
    explicit DevGuard(const ugks_ctx *c) : prev(-1), changed(0)
    {
        if (c && cudaGetDevice(&prev) == cudaSuccess && prev != c->device) changed = cudaSetDevice(c->device) == cudaSuccess;
    }
    ~DevGuard() { if (changed) cudaSetDevice(prev); }
};

static size_t al256(size_t x) { return (x + 255) & ~(size_t)255; }

// ---------------------------------------------------------------------------------------------
// Velocity-row chunks: rows are split into runs of equal sign of v (so that the upwind side of a y-face
// is uniform over a CTA), each run into equal chunks of at most `cm_target` rows; rows with v = 0 and, if the node order makes
// too many runs, everything, go to "mixed" chunks that select the side per point.  Order: [v < 0][v > 0][mixed].
constexpr int MAXCHUNK = 4096;
constexpr int MAXNV = 2048;                                          // c_v, c_wv and the chunk table of the generated kernels share the 64 KB constant bank
constexpr int MAXNU = 512;                                           // one thread per column: a CTA of <= 512 threads keeps 128 registers per thread

static void make_chunks(const double *v, int Nv, int Nu, int cm_target, KGeom *G)
{
    if (cm_target < 1) cm_target = 1;
    if ((Nu & 1) && (cm_target & 1) && cm_target > 1) cm_target -= 1;
    std::vector<int4> tmp;
    int nruns = 0;
    bool fallback = false;
    // a single v = 0 row directly followed by the v > 0 run joins that run as its first row (flag .w of its first chunk): the
    // y-fluxes of that row vanish (n = 0) and its half-range sums need one extra per-thread sum in k_cell_moments (ZROW)
    int zrow = -1;
    for (int m = 0; m + 1 < Nv; ++m)
        if (v[m] == 0.0 && v[m + 1] > 0.0 && (m == 0 || v[m - 1] < 0.0)) zrow = m;
    for (int m = 0; m < Nv && !fallback;) {
        const int sg = (v[m] > 0.0 || m == zrow) ? 1 : (v[m] < 0.0 ? -1 : 0);
        int e = m + 1;
        while (e < Nv && (v[e] > 0.0 ? 1 : (v[e] < 0.0 ? -1 : 0)) == sg) ++e;
        const int len = e - m, parts = (len + cm_target - 1) / cm_target, rows = (len + parts - 1) / parts;
        for (int p0 = m; p0 < e; p0 += rows) tmp.push_back(make_int4(p0, (p0 + rows <= e ? rows : e - p0), sg, p0 == zrow ? 1 : 0));
        m = e;
        if (++nruns > 8) fallback = true;                            // unsorted nodes: do not shred the grid
    }
    if (fallback) {
        tmp.clear();
        for (int m = 0; m < Nv; m += cm_target) tmp.push_back(make_int4(m, (m + cm_target <= Nv ? cm_target : Nv - m), 0, 0));
    }
    G->chunks.clear(); G->cmax = 0;
    const int order[3] = { -1, 1, 0 };
    int cnt[3] = { 0, 0, 0 };
    for (int o = 0; o < 3; ++o)
        for (const int4 &t : tmp)
            if (t.z == order[o]) { G->chunks.push_back(t); cnt[o]++; if (t.y > G->cmax) G->cmax = t.y; }
    G->nneg = cnt[0]; G->npos = cnt[1]; G->nmix = cnt[2];
}

// R rows in parallel (threads = Nu*R rounded up to a warp multiple), NPT = ceil(cmax / R) <= 16 points per thread: maximise
// lane use x point-slot use x a measured preference for the points per thread (the per-cell fixed work of a thread -- the
// reduction stages of k_cell_moments, the flux-column set-up of k_flux_update -- is amortised over NPT points, registers
// grow with NPT): k_cell_moments runs best at 7..8 (C3: R = 2, C4: R = 3), k_flux_update at 5..7 (C3: R = 2, C4: R = 4).
static void choose_R(int kind, int Nu, int cmax, int *R, int *npt)
{
    int best = 1; double bestscore = -1.0;
    for (int r = 1; r <= cmax && Nu * r <= (Nu > 256 ? MAXNU : 256); ++r) {
        const int n = (cmax + r - 1) / r;
        if (n > 16) continue;
        const int T = (Nu * r + 31) / 32 * 32;
        double pref;
        if (kind == JIT_MOMENTS) pref = n >= 6 && n <= 8 ? 1.0 : (n > 8 ? 0.97 : (n == 5 ? 0.8 : 0.7));
        else pref = n >= 5 && n <= 7 ? 1.0 : (n > 7 ? 0.9 : (n >= 3 ? 0.9 : 0.75));     // n = 3: M4-69 (69 columns, 9-row chunks) runs R = 3 24 % faster than R = 2
        const double score = ((double)Nu * r / T) * ((double)cmax / (r * n)) * pref;
        if (score > bestscore + 1e-9) { bestscore = score; best = r; }
    }
    *R = best; *npt = (cmax + best - 1) / best;
}

// the column ranges by sign of u (sorted nodes): a compile-time constant of k_cell_moments' stage 3
static void set_u_ranges(UgksParams &T, const double *uhost)
{
    bool sorted = true;
    for (int k = 1; k < T.Nu; ++k) if (uhost[k] < uhost[k - 1]) sorted = false;
    T.kxm_end = T.Nu; T.kxp_begin = 0;
    if (sorted) {
        int k0 = 0, k1 = 0;
        while (k0 < T.Nu && uhost[k0] < 0.0) ++k0;                   // first u >= 0
        k1 = k0; while (k1 < T.Nu && uhost[k1] <= 0.0) ++k1;         // first u > 0
        T.kxp_begin = k0; T.kxm_end = k1;
    }
}
// default launch geometry of kernel `kind` for the sizes, node signs and options (tangential) in T: the largest chunk of at
// most the target rows whose CTA fits the 227 KB of shared memory
static void choose_geometry(int kind, const UgksParams &T, const double *v, KGeom *G)
{
    const int Nu = T.Nu;
    int cm = 800 / Nu; if (cm < 1) cm = 1; if (cm > 56) cm = 56;
    if (Nu > 128) cm = kind == JIT_MOMENTS ? 14 : 5;                 // wide rows: one thread per column (measured, C5)
    else if (kind == JIT_UPDATE && cm > 1) {
        // k_flux_update: among the targets of 400 .. 800 points per chunk take the one whose CTAs waste the fewest (thread, point)
        // slots -- rows of all chunks over chunks x R x NPT, times the lanes in use.  The sweeps at the end of round 2 (M2-49, M3-49,
        // M4-49: 9-row chunks at R = 3 / NPT = 3 fill 91 % of their slots and run 10-18 % faster than the 13-row chunks of the
        // 800-point target, which fill 82 %); every other measured grid keeps its chunking (C4 20 rows, 28^2 14, 29^2 15, 69^2 9).
        int best = cm; double besteff = -1.0;
        for (int t = cm; t >= 1 && t * Nu >= 400; --t) {
            make_chunks(v, T.Nv, Nu, t, G);
            if (G->nmix > 0) { best = cm; break; }                   // unsorted nodes: keep the target
            choose_R(kind, Nu, G->cmax, &G->R, &G->npt);
            int rows = 0;
            for (const int4 &c : G->chunks) rows += c.y;
            const int th = (Nu * G->R + 31) / 32 * 32;
            const double eff = (double)rows / ((double)G->nchunk() * G->R * G->npt) * ((double)Nu * G->R / th);
            if (eff > besteff + 0.02) { besteff = eff; best = t; }  // a finer chunking has to win by 2 %
        }
        cm = best;
    }
    for (; cm >= 1; --cm) {
        make_chunks(v, T.Nv, Nu, cm, G);
        choose_R(kind, Nu, G->cmax, &G->R, &G->npt);
        if (jit_smem(kind, T, *G) <= 227 * 1024) break;
    }
    G->strip = 0;                                                    // 0 = automatic (default_strip / choose_strip in apply_geometry)
}

static int default_strip(int I) { const int ns = (I + 31) / 32; return (I + ns - 1) / ns; }     // balanced strips of <= 32 cells

// Cells per CTA march.  A march of s cells costs about s + 3 cell times (pipeline fill, the extra stencil rows), so long
// strips amortise best -- but the CTAs of a launch run in waves of (CTAs per SM) x (SMs), and on paper-sized meshes a launch
// is only a few waves: then the serial march of a CTA and the partly filled last wave decide (M4-29 at s = 32: 800 CTAs
// against 740 resident; measured 0.315 ms per step against 0.255 at s = 8).  Rule from the sweeps (C1, C2, M4-29, M3-49,
// M4-69): the longest balanced strip of at most 32 cells that still gives 4 waves, not below 8 cells (4 when even that
// leaves the GPU under one wave).
static int choose_strip(int I, int J, int nchunk, int ctas_per_sm, int sms, int s0)
{
    const long cap = (long)ctas_per_sm * sms, per_column = (long)J * nchunk;
    long ns = (4 * cap + per_column - 1) / per_column;               // strips per row for 4 waves
    if (ns < 1) ns = 1;
    int s = (int)((I + ns - 1) / ns);
    if (s >= s0) return s0;
    const int smin = per_column * ((I + 7) / 8) < cap ? 4 : 8;
    if (s < smin) s = smin;
    if (s > I) s = I;
    const int nsb = (I + s - 1) / s;                                 // balance the strips
    return (I + nsb - 1) / nsb;
}

struct Layout {
    size_t f[2], W[2], cmom, frec[2], fw[2], crec, respart, res, status, u, wu, v, wv, ghost, wallg, Wb, wallG, ghostmom,
        chunks, bcprim, Wf, total;
    int Npad, resblocks, NuP, NvP, frs, crs, nchunk_alloc;
};
// nodes and weights become literals of the generated kernel source and decide the chunking: NaN / Inf are refused up front
static bool all_finite(const double *a, int n)
{
    for (int i = 0; i < n; ++i) if (!isfinite(a[i])) return false;
    return true;
}
static bool vgrid_finite(const ugks_vgrid *vg)
{
    return all_finite(vg->u, vg->Nu) && all_finite(vg->wu, vg->Nu) && all_finite(vg->v, vg->Nv) && all_finite(vg->wv, vg->Nv);
}
// __constant__ bytes of a generated kernel: c_u, c_wu, c_v, c_wv and the chunk table; the bank holds 64 KB
static size_t jit_const_bytes(const UgksParams &T, const KGeom &G) { return 16 * ((size_t)T.Nu + T.Nv) + 16 * (size_t)G.nchunk(); }
static int make_layout(const ugks_mesh *m, const ugks_vgrid *vg, Layout *L)
{
    if (!m || !vg || m->I < 2 || m->J < 2 || vg->Nu < 1 || vg->Nu > MAXNU || vg->Nv < 1 || vg->Nv > MAXNV) return 1;
    const size_t cells = (size_t)m->I * m->J, N = (size_t)vg->Nu * vg->Nv;
    const size_t Npad = (N + 15) & ~(size_t)15;
    const size_t nfx = (size_t)(m->I + 1) * m->J, nfy = (size_t)m->I * (m->J + 1);
    L->NuP = (vg->Nu + 1) & ~1; L->NvP = (vg->Nv + 1) & ~1;
    L->frs = FR_NCOEF + L->NuP + L->NvP; L->crs = CR_NCOEF + 2 * L->NuP + 2 * L->NvP;
    // the moment buffer holds the chunks of the default geometry (the "chunk_m" tuning option may only coarsen it)
    if (!vg->v) return 1;
    if (!vg->u) return 1;
    size_t nchunk = 0;
    for (int tg = 0; tg < 2; ++tg) {                                 // room for the chunking with and without option "tangential"
        UgksParams T;
        memset(&T, 0, sizeof T);
        T.I = m->I; T.J = m->J; T.Nu = vg->Nu; T.Nv = vg->Nv; T.NuP = L->NuP; T.NvP = L->NvP; T.frs = L->frs; T.crs = L->crs; T.tangential = tg;
        set_u_ranges(T, vg->u);
        KGeom G;
        choose_geometry(JIT_MOMENTS, T, vg->v, &G);
        if ((size_t)G.nchunk() > nchunk) nchunk = (size_t)G.nchunk();
        KGeom Gu;
        choose_geometry(JIT_UPDATE, T, vg->v, &Gu);
        if (jit_const_bytes(T, G) > 65536 || jit_const_bytes(T, Gu) > 65536) return 1;   // ugks_init could not compile its kernels
    }
    if (nchunk < 1 || nchunk > MAXCHUNK) return 1;
    L->nchunk_alloc = (int)nchunk;
    L->Npad = (int)Npad;
    L->resblocks = (int)((cells + 127) / 128);
    size_t o = 0;
#define TAKE(field, bytes) do { L->field = o; o += al256(bytes); } while (0)
    TAKE(f[0], cells * Npad * 8); TAKE(f[1], cells * Npad * 8);
    TAKE(W[0], cells * 32); TAKE(W[1], cells * 32);
    TAKE(cmom, cells * nchunk * CMS * 8);
    TAKE(frec[0], nfx * L->frs * 8); TAKE(frec[1], nfy * L->frs * 8);
    TAKE(fw[0], nfx * 32); TAKE(fw[1], nfy * 32);
    TAKE(crec, cells * L->crs * 8);
    TAKE(respart, (size_t)L->resblocks * 64);
    TAKE(res, 64); TAKE(status, 64);
    TAKE(u, vg->Nu * 8); TAKE(wu, vg->Nu * 8); TAKE(v, vg->Nv * 8); TAKE(wv, vg->Nv * 8);
    TAKE(ghost, 4 * Npad * 8); TAKE(wallg, 4 * Npad * 8);
    TAKE(Wb, 128); TAKE(wallG, 128); TAKE(ghostmom, 4 * NRAW * 8); TAKE(bcprim, 128);
    TAKE(chunks, (size_t)MAXCHUNK * sizeof(int4));
    TAKE(Wf, cells * 32);
#undef TAKE
    L->total = o;
    return 0;
}

// is G a launchable geometry of kernel `kind`?  returns a message if not
static const char *check_geometry(int kind, const UgksParams &T, const KGeom &G)
{
    if (G.nchunk() < 1 || G.nchunk() > MAXCHUNK) return "bad chunk count";
    if (G.npt < 1 || G.npt > 16 || G.R < 1 || T.Nu * G.R > MAXNU || G.R * G.npt < G.cmax) return "R / points per thread out of range";
    if (G.strip < 0 || G.strip > T.I) return "strip out of range (0 = automatic, else 1..I)";
    if (jit_smem(kind, T, G) > 227 * 1024) return "chunk does not fit in shared memory";
    if (jit_const_bytes(T, G) > 65536) return "velocity nodes, weights and chunk table exceed the 64 KB constant bank";
    return nullptr;
}

// install a launch geometry of one kernel in the context: checks buffers and shared memory, compiles / fetches the kernel of
// this geometry; for k_cell_moments also uploads the chunk table (k_face_scalars sums the moment sets over its chunks)
static int apply_geometry(ugks_ctx *c, int kind, const KGeom &G)
{
    UgksParams T = c->P;
    if (kind == JIT_MOMENTS && G.nchunk() > c->nchunk_alloc) return fail(c, UGKS_EINVAL, "%s", "too many chunks for the allocated moment buffer");
    if (const char *why = check_geometry(kind, T, G)) return fail(c, UGKS_EINVAL, "%s", why);
    CK(cudaStreamSynchronize(c->st), "apply_geometry");
    if (c->gst) cudaStreamSynchronize(c->gst);
    drop_graph(c);
    JitKernel *jk = nullptr;
    char msg[240];
    KGeom Gs = G;
    const bool auto_strip = Gs.strip == 0;
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device);
    // automatic strip (few waves on small meshes, choose_strip): first from the occupancy the kernel is compiled FOR (launch bounds:
    // known on the host), so that one compile suffices; the compiled kernel's own occupancy then has the last word -- only if
    // it asks for another strip is the kernel compiled a second time
    if (auto_strip) Gs.strip = choose_strip(T.I, T.J, G.nchunk(), jit_ctas_estimate(kind, T, G), sms, default_strip(T.I));
    if (jit_get(kind, T, Gs, c->uhost, c->wuhost, c->vhost, c->wvhost, &jk, msg, sizeof msg)) return fail(c, UGKS_ECUDA, "%s", msg);
    if (auto_strip) {
        const int s = choose_strip(T.I, T.J, G.nchunk(), jit_ctas_per_sm(jk), sms, default_strip(T.I));
        if (s != Gs.strip) {
            jit_release(jk);
            Gs.strip = s;
            if (jit_get(kind, T, Gs, c->uhost, c->wuhost, c->vhost, c->wvhost, &jk, msg, sizeof msg)) return fail(c, UGKS_ECUDA, "%s", msg);
        }
    }
    const KGeom &G2 = Gs;
#ifdef UGKS_DEVELOPER
    if (getenv("UGKS_DEBUG"))
        fprintf(stderr, "ugks: %s geometry: %d chunks (cmax %d), R %d, %d points/thread, strip %d, %d CTAs/SM, %d threads, %zu B smem\n",
                kind == JIT_MOMENTS ? "k_cell_moments" : "k_flux_update", G.nchunk(), G.cmax, G.R, G.npt, G2.strip, jit_ctas_per_sm(jk), jk->threads,
                jit_smem(kind, T, G));
#endif
    if (kind == JIT_MOMENTS) {
        // the moment buffer is laid out per chunk, and k_face_scalars reads entries that k_cell_moments never writes (of the y- set
        // of the chunk that holds a v = 0 row only M00, M01, M02 are stored; the T sums without option "tangential"): they must be
        // zero, so a new chunking starts from a zeroed buffer, as ugks_init does
        CK(cudaMemsetAsync(c->P.cmom, 0, c->cells * (size_t)c->nchunk_alloc * CMS * 8, c->st), "apply_geometry");
        CK(cudaMemcpy(c->chunks_dev, G.chunks.data(), sizeof(int4) * G.nchunk(), cudaMemcpyHostToDevice), "apply_geometry");
        T.nchunk = G.nchunk(); T.nneg = G.nneg; T.npos = G.npos; T.nmix = G.nmix; T.cmax = G.cmax; T.R = G.R; T.npt = G.npt; T.strip = G2.strip;
        c->P = T;
        *c->gm = G2; jit_release(c->km); c->km = jk;
    } else { *c->gu = G2; jit_release(c->ku); c->ku = jk; }
    return UGKS_OK;
}

extern "C" {

const char *ugks_version(void) { return "ugks-b200 0.2 (sm_100a, fp64, NVRTC-specialised kernels)"; }
const char *ugks_last_error(const ugks_ctx *c) { return c ? c->err : g_err; }

int ugks_jit_check(const ugks_mesh *m, const ugks_vgrid *vg, const ugks_bcs *bcs, char *log, size_t log_bytes)
{
    if (log && log_bytes) log[0] = 0;
    Layout L;
    if (!bcs || make_layout(m, vg, &L) || !vg->u || !vg->wu || !vg->wv) return fail(nullptr, UGKS_EINVAL, "%s", "invalid mesh or velocity grid");
    if (!vgrid_finite(vg)) return fail(nullptr, UGKS_EINVAL, "%s", "velocity nodes and weights must be finite");
    UgksParams T;
    memset(&T, 0, sizeof T);
    T.I = m->I; T.J = m->J; T.Nu = vg->Nu; T.Nv = vg->Nv; T.N = vg->Nu * vg->Nv; T.Npad = L.Npad;
    T.NuP = L.NuP; T.NvP = L.NvP; T.frs = L.frs; T.crs = L.crs;
    const ugks_bc *b[4] = { &bcs->xmin, &bcs->xmax, &bcs->ymin, &bcs->ymax };
    for (int s = 0; s < 4; ++s) T.bc[s] = b[s]->type;
    set_u_ranges(T, vg->u);
#ifdef UGKS_DEVELOPER
    if (const char *e = getenv("UGKS_JIT_CHECK_TANGENTIAL")) T.tangential = atoi(e) != 0;      // check the TG variants
#endif
    std::string all;
    for (int kind = 0; kind < 2; ++kind) {
        KGeom G;
        choose_geometry(kind, T, vg->v, &G);
        G.strip = default_strip(T.I);
        if (const char *why = check_geometry(kind, T, G)) return fail(nullptr, UGKS_EINVAL, "%s", why);
        std::vector<char> cubin;
        std::string out;
        const int rc = jit_compile(kind, jit_prelude(kind, T, G, vg->u, vg->wu, vg->v, vg->wv), &cubin, &out, true);
        all += out;
        if (log && log_bytes) snprintf(log, log_bytes, "%s", all.c_str());
        if (rc) return fail(nullptr, UGKS_ECUDA, "JIT compile failed: %.200s", out.c_str());
    }
    return UGKS_OK;
}

size_t ugks_workspace_bytes(const ugks_mesh *m, const ugks_vgrid *vg)
{
    Layout L;
    return make_layout(m, vg, &L) ? 0 : L.total;
}

int ugks_init(ugks_ctx **out, const ugks_mesh *m, const ugks_vgrid *vg, const ugks_gas *gas, const ugks_bcs *bcs,
              double cfl, void *workspace_dev, size_t workspace_bytes, void *cuda_stream)
{
    ugks_ctx *c = nullptr;
    if (!out) return fail(c, UGKS_EINVAL, "%s", "out is NULL");
    *out = nullptr;
    if (!m || !vg || !gas || !bcs || !workspace_dev) return fail(c, UGKS_EINVAL, "%s", "NULL argument");
    Layout L;
    if (make_layout(m, vg, &L)) return fail(c, UGKS_EINVAL, "%s", "invalid mesh or velocity grid size (I,J >= 2; 1 <= Nu <= 512; 1 <= Nv <= 2048)");
    if (!(m->x1 > m->x0) || !(m->y1 > m->y0)) return fail(c, UGKS_EINVAL, "%s", "empty domain");
    if (!vg->u || !vg->wu || !vg->v || !vg->wv) return fail(c, UGKS_EINVAL, "%s", "NULL velocity arrays");
    if (!vgrid_finite(vg)) return fail(c, UGKS_EINVAL, "%s", "velocity nodes and weights must be finite");
    if (gas->Pr != 1.0) return fail(c, UGKS_EINVAL, "%s", "Pr must be 1 (BGK)");
    if (gas->K_int != 0) return fail(c, UGKS_EINVAL, "%s", "K_int must be 0");
    if (!(cfl > 0.0)) return fail(c, UGKS_EINVAL, "%s", "cfl must be positive");
    const ugks_bc *b[4] = { &bcs->xmin, &bcs->xmax, &bcs->ymin, &bcs->ymax };
    for (int s = 0; s < 4; ++s) {
        if (b[s]->type < 0 || b[s]->type > 2) return fail(c, UGKS_EINVAL, "%s", "unknown boundary type");
        if (b[s]->type != UGKS_BC_PERIODIC && !(b[s]->T > 0.0)) return fail(c, UGKS_EINVAL, "%s", "boundary T must be positive");
        if (b[s]->type == UGKS_BC_FIXED && !(b[s]->rho > 0.0)) return fail(c, UGKS_EINVAL, "%s", "boundary rho must be positive");
    }
    if ((b[0]->type == UGKS_BC_PERIODIC) != (b[1]->type == UGKS_BC_PERIODIC) ||
        (b[2]->type == UGKS_BC_PERIODIC) != (b[3]->type == UGKS_BC_PERIODIC))
        return fail(c, UGKS_EINVAL, "%s", "periodic sides must be paired");
    double swu = 0, swv = 0, umax = 0, vmax = 0;
    for (int k = 0; k < vg->Nu; ++k) { swu += vg->wu[k]; umax = fmax(umax, fabs(vg->u[k])); }
    for (int k = 0; k < vg->Nv; ++k) { swv += vg->wv[k]; vmax = fmax(vmax, fabs(vg->v[k])); }
    if (!(swu > 0.0) || !(swv > 0.0) || !(umax + vmax > 0.0)) return fail(c, UGKS_EINVAL, "%s", "velocity weights/nodes degenerate");
    if (workspace_bytes < L.total) return fail(c, UGKS_ENOMEM, "%s", "workspace smaller than ugks_workspace_bytes()");
    if (((uintptr_t)workspace_dev & 255) != 0) return fail(c, UGKS_EINVAL, "%s", "workspace must be 256-byte aligned");

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(c, UGKS_ECUDA, "%s", "no CUDA device: libugks has no CPU fallback");
    }
    c = (ugks_ctx *)calloc(1, sizeof *c);
    if (!c) return fail(nullptr, UGKS_ENOMEM, "%s", "host allocation failed");
    UgksParams &P = c->P;
    P.I = m->I; P.J = m->J; P.Nu = vg->Nu; P.Nv = vg->Nv; P.N = vg->Nu * vg->Nv; P.Npad = L.Npad;
    P.dx = (m->x1 - m->x0) / m->I; P.dy = (m->y1 - m->y0) / m->J;
    P.dt = cfl / (umax / P.dx + vmax / P.dy);                                   // AMB-6
    P.omega = gas->omega;
    if (gas->mu_ref > 0.0) P.mu_ref = gas->mu_ref;
    else {                                                                        // AMB-7, alpha = 1
        const double al = 1.0;
        P.mu_ref = 5.0 * (al + 1.0) * (al + 2.0) * sqrt(UGKS_PI) / (4.0 * al * (5.0 - 2.0 * gas->omega) * (7.0 - 2.0 * gas->omega)) * gas->Kn;
    }
    if (!(P.mu_ref > 0.0)) { free(c); return fail(nullptr, UGKS_EINVAL, "%s", "mu_ref / Kn must be positive"); }
    for (int s = 0; s < 4; ++s) P.bc[s] = b[s]->type;
    {   // equally spaced nodes (to 4 ulp of the largest node)?  then k_tables runs its exponentials as a two-term recurrence
        auto spacing = [](const double *x, int n) {
            if (n < 3) return 0.0;
            const double h = (x[n - 1] - x[0]) / (n - 1);
            double mx = 0.0, dev = 0.0;
            for (int k = 0; k < n; ++k) { mx = fmax(mx, fabs(x[k])); dev = fmax(dev, fabs(x[k] - (x[0] + k * h))); }
            return (h > 0.0 && dev <= 4.0 * 2.220446049250313e-16 * mx) ? h : 0.0;
        };
        P.hu = spacing(vg->u, vg->Nu); P.hv = spacing(vg->v, vg->Nv);
    }
    char *base = (char *)workspace_dev;
    auto D = [&](size_t off) { return (double *)(base + off); };
    P.f[0] = D(L.f[0]); P.f[1] = D(L.f[1]); P.W[0] = D(L.W[0]); P.W[1] = D(L.W[1]);
    P.cmom = D(L.cmom); P.frec[0] = D(L.frec[0]); P.frec[1] = D(L.frec[1]);
    P.fw[0] = D(L.fw[0]); P.fw[1] = D(L.fw[1]); P.crec = D(L.crec); P.respart = D(L.respart);
    P.NuP = L.NuP; P.NvP = L.NvP; P.frs = L.frs; P.crs = L.crs;
    P.status = (int *)(base + L.status);
    P.u = D(L.u); P.wu = D(L.wu); P.v = D(L.v); P.wv = D(L.wv);
    c->ghost = D(L.ghost); c->wallg = D(L.wallg); c->Wb = D(L.Wb); c->wallG = D(L.wallG); c->ghostmom = D(L.ghostmom);
    P.ghost = c->ghost; P.wallg = c->wallg; P.Wb = c->Wb; P.wallG = c->wallG; P.ghostmom = c->ghostmom;
    c->chunks_dev = (int4 *)(base + L.chunks); P.chunks = c->chunks_dev;
    c->res_dev = D(L.res); c->bcprim_dev = D(L.bcprim); c->Wf_dev = D(L.Wf);
    c->resblocks = L.resblocks; c->nchunk_alloc = L.nchunk_alloc;
    c->vhost = (double *)malloc(sizeof(double) * 2 * (vg->Nv + vg->Nu));      // one block: v, wv, u, wu
    if (!c->vhost) { free(c); return fail(nullptr, UGKS_ENOMEM, "%s", "host allocation failed"); }
    c->wvhost = c->vhost + vg->Nv; c->uhost = c->wvhost + vg->Nv; c->wuhost = c->uhost + vg->Nu;
    memcpy(c->vhost, vg->v, sizeof(double) * vg->Nv); memcpy(c->wvhost, vg->wv, sizeof(double) * vg->Nv);
    memcpy(c->uhost, vg->u, sizeof(double) * vg->Nu); memcpy(c->wuhost, vg->wu, sizeof(double) * vg->Nu);
    c->cells = (size_t)m->I * m->J;
    c->st = (cudaStream_t)cuda_stream;
    c->graph_mode = -1;
    set_u_ranges(P, c->uhost);
    c->gm = new KGeom(); c->gu = new KGeom();
    KGeom G0[2];
    for (int kind = 0; kind < 2; ++kind) choose_geometry(kind, P, vg->v, &G0[kind]);
    if (cudaGetDevice(&c->device) != cudaSuccess) { cudaGetLastError(); delete c->gm; delete c->gu; free(c->vhost); free(c); return fail(nullptr, UGKS_ECUDA, "%s", "cudaGetDevice failed"); }

    double bcprim[16];
    for (int s = 0; s < 4; ++s) { bcprim[s * 4] = b[s]->rho; bcprim[s * 4 + 1] = b[s]->U; bcprim[s * 4 + 2] = b[s]->V; bcprim[s * 4 + 3] = b[s]->T; }
    cudaError_t e = cudaSuccess;
    const struct { const double *src; size_t off; size_t n; } cp[5] = {
        { vg->u, L.u, (size_t)vg->Nu }, { vg->wu, L.wu, (size_t)vg->Nu }, { vg->v, L.v, (size_t)vg->Nv },
        { vg->wv, L.wv, (size_t)vg->Nv }, { bcprim, L.bcprim, 16 } };
    for (int i = 0; i < 5 && e == cudaSuccess; ++i) e = cudaMemcpyAsync(base + cp[i].off, cp[i].src, cp[i].n * 8, cudaMemcpyHostToDevice, c->st);
    if (e == cudaSuccess) e = cudaMemsetAsync(P.f[0], 0, c->cells * P.Npad * 8, c->st);
    if (e == cudaSuccess) e = cudaMemsetAsync(P.f[1], 0, c->cells * P.Npad * 8, c->st);
    if (e == cudaSuccess) e = cudaMemsetAsync(P.status, 0, 64, c->st);
    if (e == cudaSuccess) e = cudaMemsetAsync(P.cmom, 0, c->cells * (size_t)L.nchunk_alloc * CMS * 8, c->st);
    if (e == cudaSuccess) e = cudaMemsetAsync(P.frec[0], 0, (size_t)nfaces_x(P) * P.frs * 8, c->st);
    if (e == cudaSuccess) e = cudaMemsetAsync(P.frec[1], 0, (size_t)nfaces_y(P) * P.frs * 8, c->st);
    if (e == cudaSuccess) e = cudaMemsetAsync(P.crec, 0, c->cells * (size_t)P.crs * 8, c->st);
    if (e == cudaSuccess) { c->launches += launch_setup(P, c->bcprim_dev, c->ghost, c->wallg, c->Wb, c->wallG, c->ghostmom, c->st); e = cudaGetLastError(); }
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->st);
    if (e != cudaSuccess) { int rc = cuda_fail(nullptr, e, "ugks_init"); delete c->gm; delete c->gu; free(c->vhost); free(c); return rc; }
    for (int kind = 0; kind < 2; ++kind) {
        const int rc = apply_geometry(c, kind, G0[kind]);
        if (rc) { snprintf(g_err, sizeof g_err, "%s", c->err); jit_release(c->km); jit_release(c->ku); delete c->gm; delete c->gu; free(c->vhost); free(c); return rc; }
    }
    *out = c;
    return UGKS_OK;
}

void ugks_destroy(ugks_ctx *c)
{
    if (!c) return;
    DevGuard dg(c);
    cudaStreamSynchronize(c->st);
    if (c->gst) { cudaStreamSynchronize(c->gst); drop_graph(c); cudaEventDestroy(c->gin); cudaEventDestroy(c->gout); cudaStreamDestroy(c->gst); }
    for (int i = 0; i < c->nev; ++i) cudaEventDestroy(c->ev[i]);
    free(c->ev);
    free(c->vhost);
    jit_release(c->km);
    jit_release(c->ku);
    delete c->gm;
    delete c->gu;
    free(c);
}

double ugks_dt(const ugks_ctx *c) { return c ? c->P.dt : 0.0; }
double ugks_mu_ref(const ugks_ctx *c) { return c ? c->P.mu_ref : 0.0; }
long ugks_step_count(const ugks_ctx *c) { return c ? c->steps : -1; }
long ugks_launch_count(const ugks_ctx *c) { return c ? c->launches : -1; }

int ugks_set_option(ugks_ctx *c, const char *name, int value)
{
    DevGuard dg(c);
    if (!c || !name) return fail(c, UGKS_EINVAL, "%s", "NULL argument");
    UgksParams &P = c->P;
    // launch geometry of the two f-sized kernels; a "_u" suffix addresses k_flux_update alone, no suffix both kernels
    // ("R" and "chunk_m" / "strip" re-compile the kernel they change)
    {
        const size_t len = strlen(name);
        const bool only_u = len > 2 && !strcmp(name + len - 2, "_u"), only_m = len > 2 && !strcmp(name + len - 2, "_m") && strcmp(name, "chunk_m");
        char base[32];
        snprintf(base, sizeof base, "%.*s", (int)((only_u || only_m) ? len - 2 : len), name);
        if (!strcmp(base, "strip") || !strcmp(base, "chunk") || !strcmp(base, "chunk_m") || !strcmp(base, "R")) {
            for (int kind = 0; kind < 2; ++kind) {
                if ((kind == JIT_MOMENTS && only_u) || (kind == JIT_UPDATE && only_m)) continue;
                KGeom G = kind == JIT_MOMENTS ? *c->gm : *c->gu;
                if (!strcmp(base, "strip")) { if (value < 0 || value > P.I) return fail(c, UGKS_EINVAL, "%s", "strip out of range"); G.strip = value; }
                else if (!strcmp(base, "R")) {
                    if (value < 1 || P.Nu * value > MAXNU) return fail(c, UGKS_EINVAL, "%s", "R out of range");
                    G.R = value; G.npt = (G.cmax + value - 1) / value; G.strip = 0;
                } else {                                             // re-chunk with at most `value` rows per chunk
                    if (value < 1 || value > 56) return fail(c, UGKS_EINVAL, "%s", "chunk rows out of range");
                    make_chunks(c->vhost, P.Nv, P.Nu, value, &G);
                    choose_R(kind, P.Nu, G.cmax, &G.R, &G.npt);
                    G.strip = 0;
                }
                const int rc = apply_geometry(c, kind, G);
                if (rc) return rc;
            }
            return UGKS_OK;
        }
    }
    if (!strcmp(name, "tangential")) {                               // NEXT-1 (O3t/O8t): re-compiles both kernels
        if (c->gm->nmix > 0 || c->gu->nmix > 0) return fail(c, UGKS_EINVAL, "%s", "the tangential reconstruction needs v-nodes in runs of equal sign (no mixed-sign chunks)");
        const int old = P.tangential;
        P.tangential = value != 0;
        for (int kind = 0; kind < 2; ++kind) {                       // default geometry of the new mode (the staged rows differ)
            KGeom G;
            choose_geometry(kind, P, c->vhost, &G);
            const int rc = apply_geometry(c, kind, G);
            if (rc) { P.tangential = old; return rc; }
        }
        return UGKS_OK;
    }
    if (!strcmp(name, "profile")) { c->profile = value != 0; return UGKS_OK; }
    if (!strcmp(name, "poison")) { c->poison = value != 0; drop_graph(c); return UGKS_OK; }
    if (!strcmp(name, "graph")) { c->graph_mode = value < 0 ? -1 : (value != 0); if (!c->graph_mode) drop_graph(c); return UGKS_OK; }
    return fail(c, UGKS_EINVAL, "unknown option %s", name);
}

static int check_deferred(ugks_ctx *c, const char *where)
{
    CK(cudaStreamSynchronize(c->st), where);
    CK(cudaGetLastError(), where);
    int status[2] = { 0, 0 };
    CK(cudaMemcpy(status, c->P.status, sizeof status, cudaMemcpyDeviceToHost), where);
    if (status[0]) return fail(c, UGKS_ESTATE, "%s", "non-physical state (rho <= 0, lambda <= 0 or NaN) met during ugks_step");
    return UGKS_OK;
}

int ugks_set_state(ugks_ctx *c, const double *W, const double *f, int on_dev)
{
    DevGuard dg(c);
    if (!c || !W || !f) return fail(c, UGKS_EINVAL, "%s", "NULL argument");
    const UgksParams &P = c->P;
    const cudaMemcpyKind kind = on_dev ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    c->cur = 0;
    CK(cudaMemcpyAsync(P.W[0], W, c->cells * 32, kind, c->st), "ugks_set_state(W)");
    CK(cudaMemcpy2DAsync(P.f[0], (size_t)P.Npad * 8, f, (size_t)P.N * 8, (size_t)P.N * 8, c->cells, kind, c->st), "ugks_set_state(f)");
    CK(cudaMemsetAsync(P.status, 0, 64, c->st), "ugks_set_state");
    if (!on_dev) CK(cudaStreamSynchronize(c->st), "ugks_set_state");
    c->have_state = 1; c->have_res = 0; c->steps = 0;
    return UGKS_OK;
}

static void drop_graph(ugks_ctx *c)
{
    for (int p = 0; p < 2; ++p)
        if (c->gexec[p]) { cudaGraphExecDestroy(c->gexec[p]); c->gexec[p] = nullptr; }
}

// one step of the five kernels on stream st, from state parity cur; returns the kernels launched
static long enqueue_step(ugks_ctx *c, int cur, cudaStream_t st)
{
    long n = 0;
    if (c->poison) n += launch_poison_smem(st);
    n += jit_launch_cell_moments(c->km, c->P, *c->gm, cur, st);
    n += launch_face_scalars(c->P, cur, st);
    n += launch_cell_scalars(c->P, cur, c->resblocks, st);
    n += launch_tables(c->P, st);
    if (c->poison) n += launch_poison_smem(st);
    n += jit_launch_flux_update(c->ku, c->P, *c->gu, cur, st);
    return n;
}

// Launch-bound meshes replay pairs of steps from CUDA graphs captured on an internal stream.  Both graphs (one per parity of
// the ping-pong state) are captured and instantiated by the FIRST ugks_step call of the context, however short, so that the
// instantiation never falls into a later (timed) call and a call that starts from the other parity needs no re-capture.
static bool graphs_wanted(const ugks_ctx *c)
{
    return !c->profile && (c->graph_mode == 1 || (c->graph_mode < 0 && (double)c->cells * c->P.N < 3.0e7));
}
static bool ensure_graphs(ugks_ctx *c)
{
    if (c->gexec[0] && c->gexec[1]) return true;
    if (!c->gst) {
        if (cudaStreamCreateWithFlags(&c->gst, cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->gin, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->gout, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); c->graph_mode = 0; return false; }
    }
    drop_graph(c);
    for (int p = 0; p < 2; ++p) {
        cudaGraph_t g = nullptr;
        if (cudaStreamBeginCapture(c->gst, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); c->graph_mode = 0; return false; }
        c->graph_launches = enqueue_step(c, p, c->gst) + enqueue_step(c, p ^ 1, c->gst);
        if (cudaStreamEndCapture(c->gst, &g) != cudaSuccess || !g || cudaGraphInstantiate(&c->gexec[p], g, 0) != cudaSuccess) {
            cudaGetLastError(); if (g) cudaGraphDestroy(g); c->gexec[p] = nullptr; drop_graph(c); c->graph_mode = 0; return false;
        }
        cudaGraphDestroy(g);
    }
    return true;
}
// replay n / 2 pairs of steps; returns the steps done (0 if graphs are off or capture is not possible)
static int step_by_graph(ugks_ctx *c, int n)
{
    if (!graphs_wanted(c) || !ensure_graphs(c) || n < 2) return 0;
    const int pairs = n / 2;
    if (cudaEventRecord(c->gin, c->st) != cudaSuccess || cudaStreamWaitEvent(c->gst, c->gin, 0) != cudaSuccess) { cudaGetLastError(); return 0; }
    int done = 0;
    for (int i = 0; i < pairs; ++i) {
        if (cudaGraphLaunch(c->gexec[c->cur], c->gst) != cudaSuccess) break;   // the error stays pending and surfaces in ugks_step
        ++done;
    }
    if (cudaEventRecord(c->gout, c->gst) == cudaSuccess) cudaStreamWaitEvent(c->st, c->gout, 0);
    c->launches += done * c->graph_launches;
    c->steps += 2 * done;
    return 2 * done;
}

int ugks_step(ugks_ctx *c, int n)
{
    DevGuard dg(c);
    if (!c || n < 0) return fail(c, UGKS_EINVAL, "%s", "bad argument");
    if (!c->have_state) return fail(c, UGKS_ESTATE, "%s", "ugks_step before ugks_set_state");
    {
        const int done = step_by_graph(c, n);
        n -= done;
        if (done) c->have_res = 1;
    }
    if (c->profile) {
        const int need = c->nev_used + 6 * n;
        if (need > c->nev) {
            cudaEvent_t *ne = (cudaEvent_t *)realloc(c->ev, sizeof(cudaEvent_t) * need);
            if (!ne) return fail(c, UGKS_ENOMEM, "%s", "event pool");
            c->ev = ne;
            for (int i = c->nev; i < need; ++i) CK(cudaEventCreate(&c->ev[i]), "ugks_step(profile)");
            c->nev = need;
        }
    }
    for (int s = 0; s < n; ++s) {
        cudaEvent_t *e = c->profile ? c->ev + c->nev_used : nullptr;
        if (c->poison) c->launches += launch_poison_smem(c->st);
        if (e) cudaEventRecord(e[0], c->st);
        c->launches += jit_launch_cell_moments(c->km, c->P, *c->gm, c->cur, c->st);       // R, S1, S7 sums (both directions)
        if (e) cudaEventRecord(e[1], c->st);
        c->launches += launch_face_scalars(c->P, c->cur, c->st);       // S2..S5, wall density
        if (e) cudaEventRecord(e[2], c->st);
        c->launches += launch_cell_scalars(c->P, c->cur, c->resblocks, c->st);   // U1, U2 scalars, residual partials
        if (e) cudaEventRecord(e[3], c->st);
        c->launches += launch_tables(c->P, c->st);                     // S6 / U2 separable Maxwellian factors
        if (c->poison) c->launches += launch_poison_smem(c->st);
        if (e) cudaEventRecord(e[4], c->st);
        c->launches += jit_launch_flux_update(c->ku, c->P, *c->gu, c->cur, c->st);        // R, S6, S8, U3
        if (e) { cudaEventRecord(e[5], c->st); c->nev_used += 6; }
        c->cur ^= 1;
        c->steps += 1;
    }
    CK(cudaGetLastError(), "ugks_step");
    if (n > 0) c->have_res = 1;
    return UGKS_OK;
}

int ugks_kernel_times(ugks_ctx *c, double ms[5], long counts[5])
{
    DevGuard dg(c);
    if (!c || !ms || !counts) return fail(c, UGKS_EINVAL, "%s", "NULL argument");
    CK(cudaStreamSynchronize(c->st), "ugks_kernel_times");
    for (int i = 0; i + 5 < c->nev_used; i += 6)
        for (int k = 0; k < 5; ++k) {
            float t = 0.f;
            CK(cudaEventElapsedTime(&t, c->ev[i + k], c->ev[i + k + 1]), "ugks_kernel_times");
            c->kms[k] += t; c->kcnt[k] += 1;
        }
    c->nev_used = 0;
    for (int k = 0; k < 5; ++k) { ms[k] = c->kms[k]; counts[k] = c->kcnt[k]; c->kms[k] = 0.0; c->kcnt[k] = 0; }
    return UGKS_OK;
}

int ugks_sync(ugks_ctx *c)
{
    DevGuard dg(c);
    if (!c) return fail(c, UGKS_EINVAL, "%s", "NULL context");
    return check_deferred(c, "ugks_sync");
}

int ugks_moments(ugks_ctx *c, double *W_stored, double *W_of_f, int on_dev)
{
    DevGuard dg(c);
    if (!c) return fail(c, UGKS_EINVAL, "%s", "NULL context");
    if (!c->have_state) return fail(c, UGKS_ESTATE, "%s", "no state");
    const UgksParams &P = c->P;
    const cudaMemcpyKind kind = on_dev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    if (W_stored) CK(cudaMemcpyAsync(W_stored, P.W[c->cur], c->cells * 32, kind, c->st), "ugks_moments");
    if (W_of_f) {
        c->launches += launch_moments_of_f(P, P.f[c->cur], c->Wf_dev, c->st);
        CK(cudaGetLastError(), "ugks_moments");
        CK(cudaMemcpyAsync(W_of_f, c->Wf_dev, c->cells * 32, kind, c->st), "ugks_moments");
    }
    return check_deferred(c, "ugks_moments");
}

int ugks_get_f(ugks_ctx *c, double *f, int on_dev)
{
    DevGuard dg(c);
    if (!c || !f) return fail(c, UGKS_EINVAL, "%s", "NULL argument");
    if (!c->have_state) return fail(c, UGKS_ESTATE, "%s", "no state");
    const UgksParams &P = c->P;
    const cudaMemcpyKind kind = on_dev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    CK(cudaMemcpy2DAsync(f, (size_t)P.N * 8, P.f[c->cur], (size_t)P.Npad * 8, (size_t)P.N * 8, c->cells, kind, c->st), "ugks_get_f");
    return check_deferred(c, "ugks_get_f");
}

int ugks_residual(ugks_ctx *c, double res[4])
{
    DevGuard dg(c);
    if (!c || !res) return fail(c, UGKS_EINVAL, "%s", "NULL argument");
    if (!c->have_res) return fail(c, UGKS_ESTATE, "%s", "ugks_residual before the first step");
    c->launches += launch_residual_final(c->P, c->resblocks, c->res_dev, c->st);
    CK(cudaGetLastError(), "ugks_residual");
    CK(cudaMemcpyAsync(res, c->res_dev, 32, cudaMemcpyDeviceToHost, c->st), "ugks_residual");
    return check_deferred(c, "ugks_residual");
}

}  // extern "C"
