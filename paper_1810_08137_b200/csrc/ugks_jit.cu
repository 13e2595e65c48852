// ugks_jit.cu -- run-time specialisation of the two f-sized kernels (k_cell_moments, k_flux_update).
//
// ugks_init (and every option that changes the launch geometry) generates a prelude of compile-time constants -- mesh and
// velocity-grid sizes, boundary types, chunk table, R / NPT / strip, the velocity nodes and weights as hexadecimal literals --
// and compiles csrc/ugks_jit_moments.cuh + csrc/ugks_jit_update.cuh with NVRTC for sm_100a (-lineinfo).  The cubin is loaded
// through the runtime's library API (cudaLibraryLoadData / cudaLibraryGetKernel); compiled modules are cached per process by
// their prelude, so contexts of equal geometry share one module.  There is no other path: if NVRTC or the sources are missing,
// ugks_init fails.
#include "ugks_common.cuh"
#include "ugks_jit.h"

#include <dlfcn.h>
#include <nvrtc.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <map>
#include <mutex>
#include <string>
#include <vector>

namespace {

std::mutex g_mu;
std::map<std::string, JitKernel *> g_cache;
unsigned long g_tick = 0;

// unload unused kernels, least recently used first, until at most JIT_CACHE_MAX entries remain (g_mu held)
void evict_unused()
{
    while ((int)g_cache.size() > JIT_CACHE_MAX) {
        auto victim = g_cache.end();
        for (auto it = g_cache.begin(); it != g_cache.end(); ++it)
            if (it->second->users == 0 && (victim == g_cache.end() || it->second->last_used < victim->second->last_used)) victim = it;
        if (victim == g_cache.end()) return;                        // every cached kernel is in use
        if (victim->second->lib) cudaLibraryUnload(victim->second->lib);
        delete victim->second;
        g_cache.erase(victim);
    }
}

int pad2i(int x) { return (x + 1) & ~1; }
int cdivi(int a, int b) { return (a + b - 1) / b; }

// host mirrors of MomL<MIXED>::BYTES and StageL<NY>::BYTES (the device code static_asserts that they agree)
// Environment overrides exist only in a developer build (python -m paper_1810_08137_b200.build --developer => -DUGKS_DEVELOPER):
// UGKS_NSXM, UGKS_SLICE, UGKS_JIT_DEFS (extra #define lines), UGKS_JIT_MAXREG, UGKS_JIT_DUMP (keep the cubins for cuobjdump),
// UGKS_DEBUG, UGKS_JIT_CHECK_TANGENTIAL.  The shipped library reads no environment variable.
#ifdef UGKS_DEVELOPER
const char *dev_env(const char *name) { return getenv(name); }
#else
const char *dev_env(const char *) { return nullptr; }
#endif
int nsxm() { const char *e = dev_env("UGKS_NSXM"); const int n = e ? atoi(e) : 3; return n < 2 ? 2 : (n > 4 ? 4 : n); }   // x-ring slots of k_cell_moments
int smem_mom_q(const UgksParams &P, const KGeom &G, bool mixed, int QB);
int smem_upd_q(const UgksParams &P, const KGeom &G, int ny, int QB);
bool upd_slice(const UgksParams &P, const KGeom &G);
int upd_rows(const UgksParams &P, const KGeom &G) { return G.nmix > 0 ? 4 : (P.tangential ? 6 : 3); }
// slot size of a staged chunk: MC*NU + 1 doubles rounded up to even, or to a 128-byte multiple if no resident CTA is lost to it
int qb_of(int kind, const UgksParams &P, const KGeom &G)
{
    const int q2 = pad2i(G.cmax * P.Nu + 1), q16 = (G.cmax * P.Nu + 1 + 15) & ~15;
    const int s2 = kind == JIT_MOMENTS ? smem_mom_q(P, G, G.nmix > 0, q2) : smem_upd_q(P, G, upd_rows(P, G), q2);
    const int s16 = kind == JIT_MOMENTS ? smem_mom_q(P, G, G.nmix > 0, q16) : smem_upd_q(P, G, upd_rows(P, G), q16);
    return (227 * 1024) / (s16 + 1024) == (227 * 1024) / (s2 + 1024) ? q16 : q2;
}
int smem_mom(const UgksParams &P, const KGeom &G, bool mixed) { return smem_mom_q(P, G, mixed, qb_of(JIT_MOMENTS, P, G)); }
int smem_mom_q(const UgksParams &P, const KGeom &G, bool mixed, int QB)
{
    const int BT = (P.Nu * G.R + 31) / 32 * 32;
    bool zrow = false;
    for (const int4 &c : G.chunks) if (c.w) zrow = true;
    const int nrk = P.tangential ? 18 : 13;
    const int NA = mixed ? 20 : 13 + (P.tangential ? 6 : 0) + (zrow ? 1 : 0), NC = NA + 3, ny = mixed ? 2 * nrk : nrk + (zrow ? 3 : 0);
    const int lenx = P.kxm_end > P.Nu - P.kxp_begin ? P.kxm_end : P.Nu - P.kxp_begin;
    int per = P.Nu;
    for (int q = 1; q <= P.Nu; ++q) if (2 * nrk * cdivi(lenx, q) + ny * cdivi(P.Nu, q) <= BT) { per = q; break; }
    const int nitem = 2 * nrk * cdivi(lenx, per) + ny * cdivi(P.Nu, per), NUS = P.Nu | 1, NROW = G.R * G.npt + 1;
    const int total = nsxm() * QB + 4 * QB + (G.R == 1 ? 0 : NA * BT) + pad2i(2 * NC * NUS) + pad2i(14 * NUS) + pad2i(NROW * 6) +
                      pad2i(2 * nitem) + nsxm() + 3;
    return total * 8;
}
int smem_upd(const UgksParams &P, const KGeom &G, int ny) { return smem_upd_q(P, G, ny, qb_of(JIT_UPDATE, P, G)); }
// k_flux_update stages, of the v-tables of a face / cell record, only the rows of its chunk when that saves at least 64 doubles
// per table (SLICE in ugks_jit_update.cuh)
bool upd_slice(const UgksParams &P, const KGeom &G)
{
    if (const char *e = dev_env("UGKS_SLICE")) return atoi(e) != 0;
    return P.NvP - pad2i(G.cmax + 1) >= 64;
}
int smem_upd_q(const UgksParams &P, const KGeom &G, int ny, int QB)
{
    const bool sl = upd_slice(P, G);
    const int msl = pad2i(G.cmax + 1);
    const int frs = sl ? FR_NCOEF + P.NuP + msl : P.frs, crs = sl ? CR_NCOEF + 2 * P.NuP + 2 * msl : P.crs;
    const int size = ny * QB + 3 * frs + crs;
    return (3 * QB + 2 * size) * 8 + 5 * 8;
}
// CTAs per SM for __launch_bounds__: what shared memory allows, capped so that a thread keeps at least `regs` registers
int min_blocks(int threads, int smem, int regs)
{
    int by_smem = (227 * 1024) / (smem + 1024);
    int by_regs = 65536 / (threads * regs);
    int b = by_smem < by_regs ? by_smem : by_regs;
    return b < 1 ? 1 : (b > 16 ? 16 : b);
}
int threads_of(int kind, const UgksParams &P, const KGeom &G)
{
    (void)kind;
    return (P.Nu * G.R + 31) / 32 * 32;                              // no producer warp: one thread per (column, parallel row)
}

std::string dir_of_this_library()
{
    Dl_info info;
    if (!dladdr((const void *)&jit_smem, &info) || !info.dli_fname) return ".";
    std::string p(info.dli_fname);
    const size_t s = p.rfind('/');
    return s == std::string::npos ? "." : p.substr(0, s);
}
bool read_file(const std::string &path, std::string *out)
{
    FILE *f = fopen(path.c_str(), "rb");
    if (!f) return false;
    char buf[1 << 14];
    size_t n;
    out->clear();
    while ((n = fread(buf, 1, sizeof buf, f)) > 0) out->append(buf, n);
    fclose(f);
    return true;
}

// exact hexadecimal floating literal of a finite double, built from its bits: unlike printf("%a") it does not depend on the
// host application's LC_NUMERIC (a comma radix would break the generated source)
void hex_literal(double x, char out[40])
{
    unsigned long long b;
    memcpy(&b, &x, 8);
    const int e = (int)((b >> 52) & 0x7ff);
    const unsigned long long m = b & 0xfffffffffffffULL;
    const char *sg = (b >> 63) ? "-" : "";
    if (e == 0) snprintf(out, 40, "%s0x0.%013llxp-1022", sg, m);          // zero and subnormals
    else snprintf(out, 40, "%s0x1.%013llxp%+d", sg, m, e - 1023);
}
void add_doubles(std::string &s, const char *name, const double *a, int n)
{
    char buf[40];
    s += "__constant__ double "; s += name; s += "[] = {";
    for (int i = 0; i < n; ++i) { hex_literal(a[i], buf); if (i) s += ", "; s += buf; }
    s += "};\n";
}
// the first line of a compiler log that reports an error (the log starts with ptxas info lines), else its head
std::string first_error_line(const std::string &log)
{
    size_t at = log.find("error");
    if (at == std::string::npos) return log.substr(0, 200);
    size_t b = log.rfind('\n', at), e = log.find('\n', at);
    b = b == std::string::npos ? 0 : b + 1;
    return log.substr(b, (e == std::string::npos ? log.size() : e) - b).substr(0, 200);
}

}  // namespace

size_t jit_smem(int kind, const UgksParams &P, const KGeom &G)
{
    if (kind == JIT_MOMENTS) return (size_t)smem_mom(P, G, G.nmix > 0);
    return (size_t)smem_upd(P, G, G.nmix > 0 ? 4 : (P.tangential ? 6 : 3));
}

std::string jit_prelude(int kind, const UgksParams &P, const KGeom &G, const double *u, const double *wu, const double *v, const double *wv)
{
    const int threads = threads_of(kind, P, G);
    std::string s;
    char b[256];
#define DEF(name, val) do { snprintf(b, sizeof b, "#define %s %d\n", name, (int)(val)); s += b; } while (0)
    DEF("G_I", P.I); DEF("G_J", P.J); DEF("G_NU", P.Nu); DEF("G_NV", P.Nv); DEF("G_NPAD", P.Npad); DEF("G_NUP", P.NuP); DEF("G_NVP", P.NvP);
    DEF("G_FRS", P.frs); DEF("G_CRS", P.crs);
    DEF("G_BC0", P.bc[0]); DEF("G_BC1", P.bc[1]); DEF("G_BC2", P.bc[2]); DEF("G_BC3", P.bc[3]);
    DEF("G_NCHUNK", G.nchunk()); DEF("G_NMIX", G.nmix); DEF("G_MC", G.cmax); DEF("G_R", G.R); DEF("G_NPT", G.npt); DEF("G_STRIP", G.strip);
    { int z = 0; for (const int4 &c : G.chunks) if (c.w) z = 1; DEF("G_HAS_ZROW", z); }
    DEF("G_TANGENTIAL", P.tangential ? 1 : 0); DEF("G_QB", qb_of(kind, P, G));
    DEF("G_KXM_END", P.kxm_end); DEF("G_KXP_BEGIN", P.kxp_begin); DEF("G_RAGGED", G.ragged() ? 1 : 0);
    if (kind == JIT_MOMENTS) {
        const int sm_u = smem_mom(P, G, false), sm_m = smem_mom(P, G, true);
        DEF("G_SMEM_MOM", sm_u); DEF("G_SMEM_MOMX", sm_m); DEF("G_NSXM", nsxm());
        DEF("G_MINB_MOM", min_blocks(threads, sm_u, 128)); DEF("G_MINB_MOMX", min_blocks(threads, sm_m, 128));
    } else {
        const int su3 = smem_upd(P, G, P.tangential ? 6 : 3), su4 = smem_upd(P, G, 4);
        DEF("G_SMEM_UPD3", su3); DEF("G_SMEM_UPD4", su4); DEF("G_SLICE", upd_slice(P, G) ? 1 : 0);
        DEF("G_MINB_UPD", min_blocks(threads, G.nmix > 0 ? su4 : su3, 128));
    }
#undef DEF
    s += "__constant__ int4 c_chunks[] = {";
    for (int i = 0; i < G.nchunk(); ++i) { snprintf(b, sizeof b, "%s{%d, %d, %d, %d}", i ? ", " : "", G.chunks[i].x, G.chunks[i].y, G.chunks[i].z, G.chunks[i].w); s += b; }
    s += "};\n";
    if (const char *extra = dev_env("UGKS_JIT_DEFS")) { s += extra; s += "\n"; }     // developer build only
    add_doubles(s, "c_u", u, P.Nu); add_doubles(s, "c_wu", wu, P.Nu); add_doubles(s, "c_v", v, P.Nv); add_doubles(s, "c_wv", wv, P.Nv);
    return s;
}

// compile (no device needed).  On success *cubin holds the image; log receives the NVRTC log (ptxas -v lines with verbose).
int jit_compile(int kind, const std::string &prelude, std::vector<char> *cubin, std::string *log, bool verbose)
{
    // the headers are read from disk through an include path, so that -lineinfo records their real paths (ncu --import-source)
    const std::string dir = dir_of_this_library() + "/csrc";
    std::string probe;
    if (!read_file(dir + "/ugks_jit_common.cuh", &probe)) { *log = "cannot read " + dir + "/ugks_jit_common.cuh"; return 1; }
    const std::string src = prelude + (kind == JIT_MOMENTS ? "#include \"ugks_jit_moments.cuh\"\n" : "#include \"ugks_jit_update.cuh\"\n");
    nvrtcProgram prog;
    if (nvrtcCreateProgram(&prog, src.c_str(), (dir + (kind == JIT_MOMENTS ? "/ugks_jit_generated_moments.cu" : "/ugks_jit_generated_update.cu")).c_str(), 0, nullptr, nullptr) != NVRTC_SUCCESS) { *log = "nvrtcCreateProgram failed"; return 1; }
    const std::string inc = "--include-path=" + dir;
    std::vector<const char *> opts = { "--gpu-architecture=sm_100a", "-lineinfo", "--std=c++17", "-default-device", inc.c_str() };
    if (verbose) opts.push_back("--ptxas-options=-v");
    std::string maxreg;
    if (const char *e = dev_env("UGKS_JIT_MAXREG")) { maxreg = std::string("--maxrregcount=") + e; opts.push_back(maxreg.c_str()); }   // developer build only
    const nvrtcResult rc = nvrtcCompileProgram(prog, (int)opts.size(), opts.data());
    size_t n = 0;
    nvrtcGetProgramLogSize(prog, &n);
    log->assign(n, '\0');
    if (n) { nvrtcGetProgramLog(prog, &(*log)[0]); log->resize(strlen(log->c_str())); }
    if (rc != NVRTC_SUCCESS) { nvrtcDestroyProgram(&prog); *log = std::string("NVRTC: ") + nvrtcGetErrorString(rc) + "\n" + *log; return 1; }
    nvrtcGetCUBINSize(prog, &n);
    cubin->resize(n);
    nvrtcGetCUBIN(prog, cubin->data());
    nvrtcDestroyProgram(&prog);
    if (const char *dump = dev_env("UGKS_JIT_DUMP")) {               // keep the image for cuobjdump -sass: <dump>.moments.cubin / <dump>.update.cubin
        const std::string path = std::string(dump) + (kind == JIT_MOMENTS ? ".moments.cubin" : ".update.cubin");
        if (FILE *f = fopen(path.c_str(), "wb")) { fwrite(cubin->data(), 1, cubin->size(), f); fclose(f); }
    }
    return n ? 0 : 1;
}

int jit_get(int kind, const UgksParams &P, const KGeom &G, const double *u, const double *wu, const double *v, const double *wv,
            JitKernel **out, char *err, size_t errlen)
{
    const std::string pre = jit_prelude(kind, P, G, u, wu, v, wv);
    std::string key = (kind == JIT_MOMENTS ? "M:" : "U:") + pre;
    if (const char *e = dev_env("UGKS_JIT_MAXREG")) { key += "//maxreg="; key += e; }   // changes the cubin, so it is part of the key
    std::lock_guard<std::mutex> lock(g_mu);
    JitKernel *m = nullptr;
    auto it = g_cache.find(key);
    if (it != g_cache.end()) m = it->second;
    else {
        std::vector<char> cubin;
        std::string log;
        if (jit_compile(kind, pre, &cubin, &log, false)) { snprintf(err, errlen, "JIT compile failed: %s", first_error_line(log).c_str()); return 1; }
        m = new JitKernel();
        m->image.swap(cubin);
        cudaError_t e = cudaLibraryLoadData(&m->lib, m->image.data(), nullptr, nullptr, 0, nullptr, nullptr, 0);
        if (e == cudaSuccess) e = cudaLibraryGetKernel(&m->k, m->lib, kind == JIT_MOMENTS ? "k_cell_moments" : "k_flux_update");
        if (e == cudaSuccess && kind == JIT_MOMENTS && G.nmix > 0) e = cudaLibraryGetKernel(&m->kx, m->lib, "k_cell_moments_mixed");
        if (e != cudaSuccess) { snprintf(err, errlen, "JIT load failed: %s", cudaGetErrorString(e)); delete m; return 1; }
        m->threads = threads_of(kind, P, G);
        if (kind == JIT_MOMENTS) { m->smem = smem_mom(P, G, false); m->smemx = smem_mom(P, G, true); }
        else m->smem = smem_upd(P, G, G.nmix > 0 ? 4 : (P.tangential ? 6 : 3));
        g_cache[key] = m;
    }
    m->users += 1;
    m->last_used = ++g_tick;
    evict_unused();
    // shared-memory opt-in: a function attribute of the CURRENT device, set for every context (cheap, idempotent)
    cudaError_t e = cudaFuncSetAttribute((const void *)m->k, cudaFuncAttributeMaxDynamicSharedMemorySize, m->smem);
    if (e == cudaSuccess && m->kx) e = cudaFuncSetAttribute((const void *)m->kx, cudaFuncAttributeMaxDynamicSharedMemorySize, m->smemx);
    if (e != cudaSuccess) { m->users -= 1; snprintf(err, errlen, "shared-memory opt-in failed: %s", cudaGetErrorString(e)); return 1; }
    *out = m;
    return 0;
}

void jit_release(JitKernel *m)
{
    if (!m) return;
    std::lock_guard<std::mutex> lock(g_mu);
    if (m->users > 0) m->users -= 1;
    evict_unused();
}

int jit_ctas_estimate(int kind, const UgksParams &P, const KGeom &G)
{
    const int threads = threads_of(kind, P, G);
    if (kind == JIT_MOMENTS) return min_blocks(threads, smem_mom(P, G, G.nmix > 0), 128);
    return min_blocks(threads, G.nmix > 0 ? smem_upd(P, G, 4) : smem_upd(P, G, P.tangential ? 6 : 3), 128);
}

// CTAs of this kernel that one SM holds (registers, shared memory, threads) on the current device
int jit_ctas_per_sm(const JitKernel *m)
{
    int n = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, (const void *)m->k, m->threads, (size_t)m->smem) != cudaSuccess) { cudaGetLastError(); return 1; }
    return n < 1 ? 1 : n;
}

static KArgs_h make_args(const UgksParams &P, int cur)
{
    KArgs_h a;
    a.fcur = P.f[cur]; a.fnew = P.f[cur ^ 1]; a.cmom = P.cmom; a.frec0 = P.frec[0]; a.frec1 = P.frec[1]; a.crec = P.crec;
    a.ghost = P.ghost; a.wallg = P.wallg;
    return a;
}

int jit_launch_cell_moments(const JitKernel *m, const UgksParams &P, const KGeom &G, int cur, cudaStream_t st)
{
    const int nstrip = (P.I + G.strip - 1) / G.strip;
    KArgs_h a = make_args(P, cur);
    int n = 0;
    if (G.nneg + G.npos) {
        int chunk0 = 0;
        void *args[2] = { &a, &chunk0 };
        cudaLaunchKernel((const void *)m->k, dim3(P.J * nstrip * (G.nneg + G.npos)), dim3(m->threads), args, m->smem, st);
        ++n;
    }
    if (G.nmix) {
        int chunk0 = G.nneg + G.npos;
        void *args[2] = { &a, &chunk0 };
        cudaLaunchKernel((const void *)m->kx, dim3(P.J * nstrip * G.nmix), dim3(m->threads), args, m->smemx, st);
        ++n;
    }
    return n;
}

int jit_launch_flux_update(const JitKernel *m, const UgksParams &P, const KGeom &G, int cur, cudaStream_t st)
{
    const int nstrip = (P.I + G.strip - 1) / G.strip;
    KArgs_h a = make_args(P, cur);
    int chunk0 = 0;
    void *args[2] = { &a, &chunk0 };
    cudaLaunchKernel((const void *)m->k, dim3(P.J * nstrip * G.nchunk()), dim3(m->threads), args, m->smem, st);
    return 1;
}
