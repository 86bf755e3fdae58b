// C-ABI of the B200-native batched ph-AFQMC local-energy library (see include/afqmc.h for the contract).
// Host logic only: argument checks, tile-shape selection, workspace ownership, kernel launches.
// Every arithmetic step of the path runs in the kernels K0..K3 included below.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/afqmc.h"
#include "common.cuh"
#include "fp64_peak.cuh"
#include "k0_setup.cuh"
#include "k1_overlap.cuh"
#include "k2_exchange.cuh"
#include "k3_assemble.cuh"
#include "k5_spin_squared.cuh"
#include "k6_greens.cuh"
#include "k7_phaseless.cuh"
#include "k8_propagate.cuh"
#include "k10_fields.cuh"
#include "k11_pack_trial.cuh"

using namespace afqmc;

namespace {

constexpr int kMaxSmem = 232448;   // 227 KB opt-in dynamic shared memory per CTA on sm_100
constexpr int kMaxAcc = 26;        // MT*NT accumulator tiles per warp (52 doubles per lane)
constexpr int kProfSets = 256;     // ring of per-call event quadruples kept while profiling

struct SpinCfg {
    int n = 0;
    int MT = 0, NT = 0, WM = 0, gT = 0, wT = 0, strips = 0, ksc = 0, nchunks = 0, nstages = 0, H = 0, LD2 = 0;
    int n_rt = 0, n_ct_max = 0;
    int ctas_per_sm = 1;                          // persistent K2 CTAs per SM (2: two half-size CTAs, epilogues overlap K loops)
    size_t k2_smem = 0, k1_smem = 0;
    OperandLayout layA{}, layB{};
    double *A = nullptr, *B = nullptr, *psi = nullptr, *ht = nullptr, *tbuf = nullptr, *xpart = nullptr;
    double *psi_im = nullptr, *ht_im = nullptr;   // complex trial only
    double *psiA = nullptr, *psiA_im = nullptr;   // psi^T as DMMA A fragments for K1's overlap product
    int nb = 0;                                   // rows of one gamma block of the A operand: n (real trial) or 2n
    bool cplx = false;                            // this spin's trial block has a non-zero imaginary part
    // dedicated force-bias path (afqmc_enable_force_bias): operands packed with n = 1, k = (i, p)
    int f_gT = 0, f_wT = 0, f_NT = 0, f_strips = 0, f_ksteps = 0, f_ksc = 0, f_nchunks = 0, f_nstages = 0, f_n_rt = 0, f_n_ct_max = 0, f_ksplit = 1, f_kps = 0;
    size_t f_smem = 0;
    OperandLayout f_layA{}, f_layB{};
    double *f_A = nullptr, *f_B = nullptr, *f_craw = nullptr;
    size_t A_bytes = 0, B_bytes = 0;
};

thread_local std::string g_create_error;

// Tuning override AFQMC_K2_PIPELINE="ksc,stages" (include/afqmc.h), read once per process.
struct PipelineOverride { bool set = false; int ksc = 0, stages = 0; };
const PipelineOverride &pipeline_override() {
    static const PipelineOverride ov = [] {
        PipelineOverride o;
        if (const char *e = std::getenv("AFQMC_K2_PIPELINE")) o.set = std::sscanf(e, "%d,%d", &o.ksc, &o.stages) == 2;
        return o;
    }();
    return ov;
}

// Tuning override AFQMC_K2_SHAPE="warps,ctas_per_sm,gT,wT" (benchmarks only): forces K2's CTA shape.
struct ShapeOverride { bool set = false; int wm = 0, ctas = 0, gT = 0, wT = 0; };
const ShapeOverride &shape_override() {
    static const ShapeOverride ov = [] {
        ShapeOverride o;
        if (const char *e = std::getenv("AFQMC_K2_SHAPE"))
            o.set = std::sscanf(e, "%d,%d,%d,%d", &o.wm, &o.ctas, &o.gT, &o.wT) == 4 && o.wm >= 1 && o.wm <= K2_MAX_WM && o.ctas >= 1 && o.ctas <= 4;
        return o;
    }();
    return ov;
}

}  // namespace

struct afqmc_ctx {
    int N = 0, n_gamma = 0, maxw = 0, ksteps = 0, num_sms = 0;
    double e0 = 0.0;
    SpinCfg sp[2];
    double *e1 = nullptr, *logdet = nullptr;
    double2 *h_walkers = nullptr;      // device staging for the host-buffer entry point
    cudaStream_t copy_stream = nullptr; // carries the beta block's host-to-device copy under alpha's kernels
    cudaEvent_t ev_first = nullptr, ev_rest = nullptr, ev_beta = nullptr;
    double *h_outE = nullptr, *h_outO = nullptr;
    int last_nw = 0;                   // walkers whose theta the handle holds (last energy or force-bias-only call)
    int last_energy_nw = 0;            // walkers whose Coulomb traces the handle holds (last energy call)
    bool fb_enabled = false;
    // propagation (afqmc_enable_propagation): one-body factor, field-GEMM operands, work buffers
    bool prop_enabled = false;
    double dt = 0.0;
    int ldE = 0, ldt = 0, p_rt_strips = 0, p_row_tiles = 0;      // pitches of E / of the working walker layout; K9 row tiling
    double *hp = nullptr, *Emat = nullptr, *Etmp[2] = {nullptr, nullptr};
    int v_strips = 0, v_n_ct = 0, v_kps = 0, v_ksc = 0, v_nchunks = 0, v_nstages = 0;
    size_t v_smem = 0;
    long long ldv = 0;
    OperandLayout v_layA{}, v_layB{};
    double *v_A = nullptr, *v_B = nullptr, *V = nullptr, *Vtri = nullptr, *fbuf = nullptr, *xbar = nullptr, *Tb[3] = {nullptr, nullptr, nullptr};
    double *lo_old = nullptr, *lo_new = nullptr;
    cudaEvent_t pev[8] = {};           // per-phase events of the last profiled afqmc_propagate
    bool pev_valid = false;
    long long launches = 0;
    bool profiling = false;
    std::vector<cudaEvent_t> ev;       // kProfSets x 4 events, created by the first afqmc_set_profiling(1)
    long long prof_calls = 0;          // energy calls recorded since profiling was enabled
    std::string err;
};

namespace {

int fail(afqmc_ctx *ctx, int code, const char *fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (ctx) ctx->err = buf; else g_create_error = buf;
    return code;
}

#define CU_TRY(ctx, call)                                                                                   \
    do {                                                                                                    \
        cudaError_t e_ = (call);                                                                            \
        if (e_ != cudaSuccess)                                                                              \
            return fail(ctx, e_ == cudaErrorMemoryAllocation ? AFQMC_ERR_ALLOC : AFQMC_ERR_CUDA, "%s: %s", #call, \
                        cudaGetErrorString(e_));                                                            \
    } while (0)

// Staging buffer of the K2 epilogue: rows stored in pairs, pitch LD2 = 1 (mod 16) doubles, odd row at +H, H = 8 (mod 16).
void k2_staging_shape(int NT, int &H, int &LD2) {
    H = 8 * NT + ((NT & 1) ? 0 : 8);
    LD2 = H + 8 * NT;
    while (LD2 % 16 != 1) ++LD2;
}

size_t k2_smem_bytes(int strips, int NT, int ksc, int nstages) {
    const size_t stage = (size_t)ksc * (strips + NT) * 256;
    int H = 0, LD2 = 0;
    k2_staging_shape(NT, H, LD2);
    return nstages * stage + (size_t)strips * 4 * LD2 * 8 + (size_t)2 * K2_MAX_WT * K2_MAX_WM * 16 + (size_t)(2 * nstages + 2) * 8 + 16;
}

// Pipeline shape for a tile: k-steps per chunk and ring depth that fit beside the whole-tile staging buffer.
bool choose_pipeline(int strips, int NT, int ksteps, size_t budget, int &ksc, int &nst) {
    if (const PipelineOverride &ov = pipeline_override(); ov.set) {
        const int kc = ov.ksc, s = ov.stages;
        if (kc >= 1 && kc <= ksteps && s >= 2 && s <= 16 && k2_smem_bytes(strips, NT, kc, s) <= budget) {
            ksc = kc; nst = s;
            return true;
        }
    }
    // Measured on cu2o2 (profiles/): with the non-blocking producer the most k-steps in flight
    // wins, and at equal depth fewer, larger chunks win (5 x 2 stages 85.4 %, 3 x 3 84.8 %, 2 x 5 84.2 % of peak).
    int best = 0;
    for (int s = 2; s <= 5; ++s) {
        for (int kc = std::min(12, std::max(2, ksteps / 10)); kc >= 1; --kc) {   // short K loops want short chunks (tile start-up)
            if (kc > ksteps) continue;
            if (k2_smem_bytes(strips, NT, kc, s) > budget) continue;
            if (kc * s > best) { best = kc * s; ksc = kc; nst = s; }
            break;
        }
    }
    return best > 0;
}

// Pick the K2 tile shape for one spin: maximise (useful rows / issued rows) x (useful cols / issued cols),
// balanced over the 4 SM sub-partitions (strip s -> warp s % WM -> sub-partition s % 4).
bool choose_cfg(int n, bool cplx, int N, int n_gamma, int maxw, SpinCfg &c) {
    c.n = n;
    const int nb = cplx ? 2 * n : n;      // rows per gamma block
    c.nb = nb;
    if (n == 0) return true;
    const int ksteps = (N + 3) / 4;
    double best = -1.0;
    // Every warp of the CTA is an MMA warp: K2_MAX_WM = 12 warps (3 per SM sub-partition) is what the register file
    // allows at 168 registers per thread, and fewer warps never scored higher in any shape.
    const ShapeOverride &so = shape_override();
    const int WM = so.set ? so.wm : K2_MAX_WM;
    c.ctas_per_sm = so.set ? so.ctas : 1;
    const size_t budget = c.ctas_per_sm == 1 ? (size_t)kMaxSmem : (size_t)(233472 / c.ctas_per_sm - 1024);
    for (int wT = 1; wT <= K2_MAX_WT; ++wT) {
        if (so.set && so.wT > 0 && wT != so.wT) continue;
        const int cols = 2 * wT * n, NT = (cols + 7) / 8;
        if (NT > 16) continue;
        const double colEff = cols / (8.0 * NT);
        for (int MT = 1; MT <= 4; ++MT) {
            if (MT * NT > kMaxAcc) continue;
            for (int gT = 1; gT <= n_gamma; ++gT) {
                const int strips = (gT * nb + 7) / 8;
                if (strips > MT * WM) break;
                if (so.set && so.gT > 0 && gT != so.gT) continue;
                if ((strips + WM - 1) / WM < MT && MT > 1) continue;   // a smaller MT covers it
                const int maxload = (strips + 3) / 4;
                const double rowEff = (gT * nb / 8.0) / (4.0 * maxload);
                int ksc = 0, nst = 0;
                if (!choose_pipeline(strips, NT, ksteps, budget, ksc, nst)) continue;
                const long long ntiles = (long long)((n_gamma + gT - 1) / gT) * ((maxw + wT - 1) / wT);
                const double fill = ntiles >= 148 ? 1.0 : ntiles / 148.0;
                const double lds = 1.0 - 0.03 * (double)(MT + NT) / (MT * NT);
                const double score = rowEff * colEff * lds * (0.5 + 0.5 * fill);
                if (score > best + 1e-12) {
                    best = score;
                    c.MT = MT; c.NT = NT; c.WM = WM; c.gT = gT; c.wT = wT; c.strips = strips;
                    c.ksc = ksc; c.nstages = nst;
                }
            }
        }
    }
    if (best < 0) return false;
    c.nchunks = (ksteps + c.ksc - 1) / c.ksc;
    c.n_rt = (n_gamma + c.gT - 1) / c.gT;
    c.n_ct_max = (maxw + c.wT - 1) / c.wT;
    c.k2_smem = k2_smem_bytes(c.strips, c.NT, c.ksc, c.nstages);
    k2_staging_shape(c.NT, c.H, c.LD2);
    c.layA = OperandLayout{n, c.strips, ksteps, c.gT, (long long)c.strips * ksteps * 32};
    c.layB = OperandLayout{n, c.NT, ksteps, c.wT, (long long)c.NT * ksteps * 32};
    c.A_bytes = (size_t)c.n_rt * c.layA.tile_doubles * 8;
    c.B_bytes = (size_t)c.n_ct_max * c.layB.tile_doubles * 8;
    c.k1_smem = (size_t)k1_layout(n, cplx).total;
    return true;
}

using K2Fn = void (*)(const K2Params);

template <int MT, int NT>
K2Fn k2_pick_nt(int nt) {
    if constexpr (NT == 0) {
        return nullptr;
    } else {
        if (nt == NT) {
            if constexpr (MT * NT <= kMaxAcc) return k2_exchange<MT, NT>;
            else return nullptr;
        }
        return k2_pick_nt<MT, NT - 1>(nt);
    }
}
K2Fn k2_pick(int mt, int nt) {
    switch (mt) {
        case 1: return k2_pick_nt<1, 16>(nt);
        case 2: return k2_pick_nt<2, 13>(nt);
        case 3: return k2_pick_nt<3, 8>(nt);
        case 4: return k2_pick_nt<4, 6>(nt);
    }
    return nullptr;
}

using K2FbFn = void (*)(const K2FbParams);
template <int NT>
K2FbFn k2_pick_fb_nt(int nt) {
    if constexpr (NT == 0) {
        return nullptr;
    } else {
        if (nt == NT) return k2_force_bias<NT>;
        return k2_pick_fb_nt<NT - 1>(nt);
    }
}
K2FbFn k2_pick_fb(int nt) { return k2_pick_fb_nt<16>(nt); }

void free_ctx(afqmc_ctx *c) {
    if (!c) return;
    for (int s = 0; s < 2; ++s) {
        cudaFree(c->sp[s].A); cudaFree(c->sp[s].B); cudaFree(c->sp[s].psi); cudaFree(c->sp[s].ht); cudaFree(c->sp[s].psi_im); cudaFree(c->sp[s].ht_im);
        cudaFree(c->sp[s].psiA); cudaFree(c->sp[s].psiA_im);
        cudaFree(c->sp[s].f_A); cudaFree(c->sp[s].f_B); cudaFree(c->sp[s].f_craw);
        cudaFree(c->sp[s].tbuf); cudaFree(c->sp[s].xpart);
    }
    cudaFree(c->e1); cudaFree(c->logdet); cudaFree(c->h_walkers); cudaFree(c->h_outE); cudaFree(c->h_outO);
    cudaFree(c->hp); cudaFree(c->Emat); cudaFree(c->Etmp[0]); cudaFree(c->Etmp[1]); cudaFree(c->v_A); cudaFree(c->v_B);
    cudaFree(c->V); cudaFree(c->Vtri); cudaFree(c->fbuf); cudaFree(c->xbar); cudaFree(c->Tb[0]); cudaFree(c->Tb[1]); cudaFree(c->Tb[2]);
    cudaFree(c->lo_old); cudaFree(c->lo_new);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    if (c->ev_first) cudaEventDestroy(c->ev_first);
    if (c->ev_rest) cudaEventDestroy(c->ev_rest);
    if (c->ev_beta) cudaEventDestroy(c->ev_beta);
    for (auto &e : c->pev) if (e) cudaEventDestroy(e);
    for (auto &e : c->ev) if (e) cudaEventDestroy(e);
    delete c;
}

// Opt a kernel in to the full 227 KB of dynamic shared memory.  The attribute is process-global per kernel, so it is
// always set to the ceiling: a smaller per-handle value would lower the cap for another spin or handle that shares
// the instantiation (the launch itself passes the exact size).
template <class Fn>
cudaError_t allow_max_smem(Fn fn) {
    cudaFuncAttributes fa{};
    if (cudaError_t e = cudaFuncGetAttributes(&fa, (const void *)fn); e != cudaSuccess) return e;
    return cudaFuncSetAttribute((const void *)fn, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                kMaxSmem - (int)fa.sharedSizeBytes);   // static + dynamic <= 227 KB
}

int check_arch(afqmc_ctx *ctx, int *num_sms) {
    int dev = 0;
    CU_TRY(ctx, cudaGetDevice(&dev));
    int major = 0, sms = 0;
    CU_TRY(ctx, cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    CU_TRY(ctx, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    if (major != 10) return fail(ctx, AFQMC_ERR_ARCH, "device compute capability %d.x is not sm_100", major);
    if (num_sms) *num_sms = sms;
    return AFQMC_OK;
}

// K1 for `n_walkers` walkers; with_fb also writes theta in the force-bias operand order.  spin = -1: both spins in one
// launch; 0 / 1: that spin only, walkers w0 .. w0 + count - 1 (the host-buffer entry point starts on the walkers that
// have arrived while the rest is still being copied).  n_walkers is always the call's total (it fixes the beta offset).
int launch_k1(afqmc_ctx *ctx, const void *walkers, int n_walkers, bool with_fb, cudaStream_t stream, int spin = -1, int w0 = 0,
              int count = -1) {
    const int N = ctx->N;
    K1Params p1{};
    p1.walkers = reinterpret_cast<const double2 *>(walkers);
    p1.n_walkers = n_walkers; p1.N = N; p1.maxw = ctx->maxw;
    p1.spin0 = spin < 0 ? 0 : spin;
    p1.w0 = w0;
    p1.spin_off[0] = 0;
    p1.spin_off[1] = (long long)n_walkers * N * ctx->sp[0].n;
    for (int s = 0; s < 2; ++s) {
        p1.n[s] = ctx->sp[s].n; p1.psiA[s] = ctx->sp[s].psiA; p1.psiA_im[s] = ctx->sp[s].psiA_im;
        p1.ht[s] = ctx->sp[s].ht; p1.ht_im[s] = ctx->sp[s].ht_im;
        p1.thetaB[s] = ctx->sp[s].B; p1.layB[s] = ctx->sp[s].layB;
        p1.thetaF[s] = with_fb ? ctx->sp[s].f_B : nullptr; p1.layF[s] = ctx->sp[s].f_layB;
    }
    p1.logdet = ctx->logdet; p1.e1 = ctx->e1;
    const bool big = std::max(ctx->sp[0].n, ctx->sp[1].n) > 32;
    const int nwl = count < 0 ? n_walkers : count, nsp = spin < 0 ? 2 : 1;
    const size_t k1s = std::max(ctx->sp[0].k1_smem, ctx->sp[1].k1_smem);
    const dim3 grid(nwl, nsp);
    // n <= 32: four CTAs per SM; larger n: two per SM when the shared memory allows it (measured at medium, n = 40:
    // 0.185 -> 0.130 ms), else one per SM with the whole register file (large, n = 50: 1.21 ms against 1.45 at 128 registers)
    const int size = !big ? 0 : (2 * (k1s + 1024) <= 233472 ? 1 : 2);
    if (size == 2) {
        if (with_fb) k1_overlap_inverse_theta<2, true><<<grid, K1_THREADS, k1s, stream>>>(p1);
        else k1_overlap_inverse_theta<2, false><<<grid, K1_THREADS, k1s, stream>>>(p1);
    } else if (size == 1) {
        if (with_fb) k1_overlap_inverse_theta<1, true><<<grid, K1_THREADS, k1s, stream>>>(p1);
        else k1_overlap_inverse_theta<1, false><<<grid, K1_THREADS, k1s, stream>>>(p1);
    } else {
        if (with_fb) k1_overlap_inverse_theta<0, true><<<grid, K1_THREADS, k1s, stream>>>(p1);
        else k1_overlap_inverse_theta<0, false><<<grid, K1_THREADS, k1s, stream>>>(p1);
    }
    CU_TRY(ctx, cudaGetLastError());
    ctx->launches += 1;
    return AFQMC_OK;
}

// The force-bias GEMM (one launch per spin) and the combine kernel, on the theta K1<with_fb> has just written.
int launch_force_bias_gemm(afqmc_ctx *ctx, int n_walkers, double *out, cudaStream_t stream) {
    K4Params p4{};
    p4.n_walkers = n_walkers; p4.n_gamma = ctx->n_gamma; p4.out = out;
    for (int s = 0; s < 2; ++s) {
        const SpinCfg &sc = ctx->sp[s];
        p4.n[s] = sc.n;
        if (sc.n == 0) continue;
        const int nbf = sc.cplx ? 2 : 1;
        K2FbParams p2{};
        p2.A = sc.f_A; p2.B = sc.f_B;
        p2.itemA_doubles = sc.f_layA.tile_doubles / sc.f_ksplit;   // parts of a tile are contiguous
        p2.tileB_doubles = sc.f_layB.tile_doubles;
        p2.partB_doubles = (long long)sc.f_kps * sc.f_NT * 32;
        p2.rows_per_tile = sc.f_gT * nbf; p2.rows_total = ctx->n_gamma * nbf;
        p2.strips = sc.f_strips; p2.WM = K2_MAX_WM;
        p2.kps = sc.f_kps; p2.ksc = sc.f_ksc; p2.nchunks = sc.f_nchunks; p2.nstages = sc.f_nstages;
        p2.n_items_r = sc.f_n_rt * sc.f_ksplit; p2.ksplit = sc.f_ksplit; p2.n_ct = (n_walkers + sc.f_wT - 1) / sc.f_wT;
        p2.craw = sc.f_craw;
        const long long ntiles = (long long)p2.n_items_r * p2.n_ct;
        const int grid = (int)std::min<long long>(ntiles, ctx->num_sms);
        K2FbFn fn = k2_pick_fb(sc.f_NT);
        fn<<<grid, 32 * K2_MAX_WM, sc.f_smem, stream>>>(p2);
        CU_TRY(ctx, cudaGetLastError());
        ctx->launches += 1;
        p4.nb[s] = nbf; p4.wT[s] = sc.f_wT; p4.n_ct[s] = p2.n_ct; p4.ldc[s] = sc.f_NT * 8; p4.craw[s] = sc.f_craw; p4.ksplit[s] = sc.f_ksplit;
    }
    const long long total = (long long)n_walkers * ctx->n_gamma;
    k4_force_bias_combine<<<(unsigned)((total + 255) / 256), 256, 0, stream>>>(p4);
    CU_TRY(ctx, cudaGetLastError());
    ctx->launches += 1;
    return AFQMC_OK;
}

// One K9 launch: Out_b = alpha M_b In_b, b = 0 .. batch-1; optionally Sum_b += Out_b, or Out_b = Add_b + alpha M_b In_b.
int launch_k9(afqmc_ctx *ctx, const double *Mre, const double *Mim, long long m_stride, int ldm, const double *In, double *Out,
              double *Sum, long long io_stride, int ld, int C, int batch, double alpha, cudaStream_t stream, const double *Add = nullptr) {
    K9Params p{};
    p.Mre = Mre; p.Mim = Mim; p.m_batch_stride = m_stride; p.ldm = ldm; p.In = In; p.Out = Out; p.Sum = Sum; p.Add = Add;
    p.io_batch_stride = io_stride; p.ld = ld; p.N = ctx->N; p.C = C; p.rt_strips = ctx->p_rt_strips; p.alpha = alpha;
    // column groups: as few as fit the accumulators, of equal width (splitting further to fill the last wave of CTAs was
    // measured and lost: 5.6 vs 4.7 ms for the Taylor phase at cu2o2, the M tile is then staged twice)
    const int blocks = (C + 7) / 8;
    const int groups = (blocks + K9_NT - 1) / K9_NT;
    p.cg_blocks = (blocks + groups - 1) / groups;
    const int col_groups = (blocks + p.cg_blocks - 1) / p.cg_blocks;
    // One CTA per SM: the batch items that fill whole rounds of the GPU go in one launch with the regular row tiles; the
    // rest -- a partial round that would cost as much as a full one -- goes in a second launch with tiles of half the
    // height, which finishes in about 0.6 of a round (cu2o2: 444 + 136 CTAs instead of 512 = 3.46 waves).
    const long long per_item = (long long)ctx->p_row_tiles * col_groups;
    int main_items = batch;
    if (batch > 1 && per_item * batch > ctx->num_sms) {
        const long long rounds = per_item * batch / ctx->num_sms;
        main_items = (int)(rounds * ctx->num_sms / per_item);
    }
    const int S = (ctx->N + 7) / 8;
    if (main_items > 0) {
        k9_apply<<<dim3(ctx->p_row_tiles, col_groups, main_items), K9_THREADS, K9_SMEM, stream>>>(p);
        CU_TRY(ctx, cudaGetLastError());
        ctx->launches += 1;
    }
    if (main_items < batch) {
        K9Params t = p;
        const int tiles = std::min(S, 2 * ctx->p_row_tiles);
        t.rt_strips = (S + tiles - 1) / tiles;
        t.Mre = Mre + (long long)main_items * m_stride;
        t.Mim = Mim ? Mim + (long long)main_items * m_stride : nullptr;
        t.In = In + (long long)main_items * io_stride;
        t.Out = Out + (long long)main_items * io_stride;
        t.Sum = Sum ? Sum + (long long)main_items * io_stride : nullptr;
        t.Add = Add ? Add + (long long)main_items * io_stride : nullptr;
        k9_apply<<<dim3((S + t.rt_strips - 1) / t.rt_strips, col_groups, batch - main_items), K9_THREADS, K9_SMEM, stream>>>(t);
        CU_TRY(ctx, cudaGetLastError());
        ctx->launches += 1;
    }
    return AFQMC_OK;
}

}  // namespace

extern "C" {

int afqmc_create(const double *h1e, const double *chol, const void *trial, int N, int n_alpha, int n_beta,
                 int n_gamma, double e0, int max_walkers, void *stream_, afqmc_ctx **out) {
    if (out) *out = nullptr;
    if (!h1e || !chol || !trial || !out) return fail(nullptr, AFQMC_ERR_ARG, "afqmc_create: null pointer argument");
    if (N < 1 || n_gamma < 1 || max_walkers < 1 || n_alpha < 0 || n_beta < 0 || n_alpha > N || n_beta > N ||
        n_alpha + n_beta < 1)
        return fail(nullptr, AFQMC_ERR_ARG, "afqmc_create: size out of range (N=%d n_alpha=%d n_beta=%d n_gamma=%d max_walkers=%d)",
                    N, n_alpha, n_beta, n_gamma, max_walkers);
    if (n_alpha > AFQMC_MAX_NOCC || n_beta > AFQMC_MAX_NOCC)
        return fail(nullptr, AFQMC_ERR_UNSUPPORTED, "afqmc_create: n_sigma > %d is not supported yet", AFQMC_MAX_NOCC);
    cudaStream_t stream = (cudaStream_t)stream_;
    int sms = 0;
    if (int rc = check_arch(nullptr, &sms)) return rc;

    afqmc_ctx *c = new afqmc_ctx();
    c->N = N; c->n_gamma = n_gamma; c->maxw = max_walkers; c->e0 = e0; c->ksteps = (N + 3) / 4; c->num_sms = sms;
    const int ns[2] = {n_alpha, n_beta};
#define CR_TRY(call)                                                                                          \
    do {                                                                                                      \
        cudaError_t e_ = (call);                                                                              \
        if (e_ != cudaSuccess) {                                                                              \
            int rc_ = fail(nullptr, e_ == cudaErrorMemoryAllocation ? AFQMC_ERR_ALLOC : AFQMC_ERR_CUDA,       \
                           "afqmc_create: %s: %s", #call, cudaGetErrorString(e_));                            \
            free_ctx(c);                                                                                      \
            return rc_;                                                                                       \
        }                                                                                                     \
    } while (0)

    // trial: split into per-spin real planes [N][n].  A spin whose trial block is real ("a real-valued
    // array rchol": all of BASELINE.json's configs) gets a real Ltilde and two real DMMA products per complex T; a
    // complex block gets Ltilde = (Re, Im) stacked in every gamma block and four products.
    const size_t ntrial = (size_t)N * (n_alpha + n_beta);
    std::vector<double> trial_h(2 * ntrial);
    CR_TRY(cudaMemcpyAsync(trial_h.data(), trial, 2 * ntrial * sizeof(double), cudaMemcpyDeviceToHost, stream));
    CR_TRY(cudaStreamSynchronize(stream));
    for (size_t k = 0; k < 2 * ntrial; ++k) {
        if (!std::isfinite(trial_h[k])) {
            free_ctx(c);
            return fail(nullptr, AFQMC_ERR_ARG, "afqmc_create: trial has a non-finite entry");
        }
    }
    size_t toff = 0;
    for (int s = 0; s < 2; ++s) {
        SpinCfg &sc = c->sp[s];
        const int n = ns[s];
        bool cplx = false;
        for (size_t k = 0; k < (size_t)N * n; ++k) cplx = cplx || (trial_h[2 * (toff + k) + 1] != 0.0);
        sc.cplx = cplx;
        if (!choose_cfg(n, cplx, N, n_gamma, max_walkers, sc)) {
            free_ctx(c);
            return fail(nullptr, AFQMC_ERR_UNSUPPORTED, "afqmc_create: no K2 tile shape fits n_sigma=%d", n);
        }
        if (n == 0) continue;
        std::vector<double> psi_h((size_t)N * n), psi_ih((size_t)N * n);
        for (size_t k = 0; k < psi_h.size(); ++k) { psi_h[k] = trial_h[2 * (toff + k)]; psi_ih[k] = trial_h[2 * (toff + k) + 1]; }
        toff += (size_t)N * n;
        CR_TRY(cudaMalloc(&sc.psi, psi_h.size() * 8));
        CR_TRY(cudaMemcpyAsync(sc.psi, psi_h.data(), psi_h.size() * 8, cudaMemcpyHostToDevice, stream));
        if (cplx) {
            CR_TRY(cudaMalloc(&sc.psi_im, psi_ih.size() * 8));
            CR_TRY(cudaMemcpyAsync(sc.psi_im, psi_ih.data(), psi_ih.size() * 8, cudaMemcpyHostToDevice, stream));
            CR_TRY(cudaMalloc(&sc.ht_im, (size_t)n * N * 8));
        }
        {   // psi^T in DMMA A-fragment order for K1: [k-step][8-row strip of i][lane = r * 4 + k], p = 4 * kstep + k,
            // zero-padded to whole chunks of K1_ROWS rows of phi (k1_overlap.cuh)
            const int ns8 = (n + 7) / 8, kpad = 8 * ((N + K1_ROWS - 1) / K1_ROWS);
            std::vector<double> pa((size_t)kpad * ns8 * 32, 0.0), pai(cplx ? pa.size() : 0, 0.0);
            for (int p = 0; p < N; ++p)
                for (int i = 0; i < n; ++i) {
                    const size_t o = ((size_t)(p >> 2) * ns8 + (i >> 3)) * 32 + (i & 7) * 4 + (p & 3);
                    pa[o] = psi_h[(size_t)p * n + i];
                    if (cplx) pai[o] = psi_ih[(size_t)p * n + i];
                }
            CR_TRY(cudaMalloc(&sc.psiA, pa.size() * 8));
            CR_TRY(cudaMemcpyAsync(sc.psiA, pa.data(), pa.size() * 8, cudaMemcpyHostToDevice, stream));
            if (cplx) {
                CR_TRY(cudaMalloc(&sc.psiA_im, pai.size() * 8));
                CR_TRY(cudaMemcpyAsync(sc.psiA_im, pai.data(), pai.size() * 8, cudaMemcpyHostToDevice, stream));
            }
            CR_TRY(cudaStreamSynchronize(stream));
        }
        CR_TRY(cudaStreamSynchronize(stream));
        CR_TRY(cudaMalloc(&sc.ht, (size_t)n * N * 8));
        CR_TRY(cudaMalloc(&sc.A, sc.A_bytes));
        CR_TRY(cudaMalloc(&sc.B, sc.B_bytes));
        CR_TRY(cudaMalloc(&sc.tbuf, (size_t)max_walkers * n_gamma * 16));
        CR_TRY(cudaMalloc(&sc.xpart, (size_t)sc.n_rt * max_walkers * 16));
        CR_TRY(cudaMemsetAsync(sc.A, 0, sc.A_bytes, stream));
        CR_TRY(cudaMemsetAsync(sc.B, 0, sc.B_bytes, stream));
        CR_TRY(cudaMemsetAsync(sc.tbuf, 0, (size_t)max_walkers * n_gamma * 16, stream));
        dim3 grid(n_gamma, (N + 127) / 128);
        k0_half_rotate_h<<<(n * N + 255) / 256, 256, 0, stream>>>(h1e, sc.psi, N, n, 1.0, sc.ht);
        CR_TRY(cudaGetLastError());
        k0_half_rotate_chol<<<grid, 128, 0, stream>>>(chol, sc.psi, N, n, n_gamma, sc.nb, 0, 1.0, sc.layA, sc.A, OperandLayout{}, nullptr);
        CR_TRY(cudaGetLastError());
        c->launches += 2;
        if (cplx) {                                   // conj(psi) = Re psi - i Im psi
            k0_half_rotate_h<<<(n * N + 255) / 256, 256, 0, stream>>>(h1e, sc.psi_im, N, n, -1.0, sc.ht_im);
            CR_TRY(cudaGetLastError());
            k0_half_rotate_chol<<<grid, 128, 0, stream>>>(chol, sc.psi_im, N, n, n_gamma, sc.nb, n, -1.0, sc.layA, sc.A, OperandLayout{}, nullptr);
            CR_TRY(cudaGetLastError());
            c->launches += 2;
        }
        K2Fn fn = k2_pick(sc.MT, sc.NT);
        if (!fn) {
            free_ctx(c);
            return fail(nullptr, AFQMC_ERR_UNSUPPORTED, "afqmc_create: no K2 instantiation for MT=%d NT=%d", sc.MT, sc.NT);
        }
        CR_TRY(allow_max_smem(fn));
    }
    CR_TRY(allow_max_smem(k1_overlap_inverse_theta<0, false>));
    CR_TRY(allow_max_smem(k1_overlap_inverse_theta<0, true>));
    CR_TRY(allow_max_smem(k1_overlap_inverse_theta<1, false>));
    CR_TRY(allow_max_smem(k1_overlap_inverse_theta<1, true>));
    CR_TRY(allow_max_smem(k1_overlap_inverse_theta<2, false>));
    CR_TRY(allow_max_smem(k1_overlap_inverse_theta<2, true>));
    CR_TRY(allow_max_smem(k5_spin_squared));
    CR_TRY(allow_max_smem(k6_greens_function));
    CR_TRY(cudaMalloc(&c->e1, (size_t)2 * max_walkers * 16));
    CR_TRY(cudaMalloc(&c->logdet, (size_t)2 * max_walkers * 16));
    CR_TRY(cudaMemsetAsync(c->e1, 0, (size_t)2 * max_walkers * 16, stream));
    CR_TRY(cudaMemsetAsync(c->logdet, 0, (size_t)2 * max_walkers * 16, stream));
    CR_TRY(cudaMalloc(&c->h_walkers, (size_t)max_walkers * N * (n_alpha + n_beta) * 16));
    CR_TRY(cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
    CR_TRY(cudaEventCreateWithFlags(&c->ev_first, cudaEventDisableTiming));
    CR_TRY(cudaEventCreateWithFlags(&c->ev_rest, cudaEventDisableTiming));
    CR_TRY(cudaEventCreateWithFlags(&c->ev_beta, cudaEventDisableTiming));
    CR_TRY(cudaMalloc(&c->h_outE, (size_t)max_walkers * 16));
    CR_TRY(cudaMalloc(&c->h_outO, (size_t)max_walkers * 16));
    CR_TRY(cudaStreamSynchronize(stream));
#undef CR_TRY
    *out = c;
    return AFQMC_OK;
}

// One K2 launch: spin s, walkers w0 .. w0 + count - 1 (w0 a multiple of the tile's walker count).
static int launch_k2(afqmc_ctx *ctx, int s, int w0, int count, cudaStream_t stream) {
    const SpinCfg &sc = ctx->sp[s];
    K2Params p2{};
    p2.A = sc.A; p2.B = sc.B + (long long)(w0 / sc.wT) * sc.layB.tile_doubles;
    p2.tileA_doubles = sc.layA.tile_doubles; p2.tileB_doubles = sc.layB.tile_doubles;
    p2.n = sc.n; p2.nb = sc.nb; p2.cplx = sc.cplx ? 1 : 0; p2.gT = sc.gT; p2.wT = sc.wT; p2.strips = sc.strips; p2.WM = sc.WM;
    p2.ksteps = ctx->ksteps; p2.ksc = sc.ksc; p2.nchunks = sc.nchunks; p2.nstages = sc.nstages;
    p2.n_rt = sc.n_rt; p2.n_ct = (count + sc.wT - 1) / sc.wT;
    p2.n_gamma = ctx->n_gamma; p2.n_walkers = count; p2.maxw = ctx->maxw; p2.H = sc.H; p2.LD2 = sc.LD2;
    p2.tbuf = sc.tbuf + (long long)w0 * ctx->n_gamma * 2; p2.xpart = sc.xpart + (long long)w0 * 2;
    const long long ntiles = (long long)p2.n_rt * p2.n_ct;
    const int grid = (int)std::min<long long>(ntiles, (long long)ctx->num_sms * sc.ctas_per_sm);
    K2Fn fn = k2_pick(sc.MT, sc.NT);
    fn<<<grid, 32 * sc.WM, sc.k2_smem, stream>>>(p2);
    CU_TRY(ctx, cudaGetLastError());
    ctx->launches += 1;
    return AFQMC_OK;
}

// A piece of an energy call: K1 and K2 of one spin on a range of walkers, after an optional event (the host-buffer entry
// point records one per block of walkers it copies on its own stream).
struct EnergyPiece { int spin, w0, count; cudaEvent_t wait; };

// K1 -> K2 -> K3 on `stream`.  Without pieces: K1 for both spins in one launch, then K2 once per spin.
static int run_energy(afqmc_ctx *ctx, const void *walkers, int n_walkers, void *out_energies, void *out_overlaps,
                      cudaStream_t stream, const EnergyPiece *pieces, int n_pieces) {
    cudaEvent_t *ev = ctx->profiling ? &ctx->ev[(size_t)(ctx->prof_calls % kProfSets) * 4] : nullptr;
    if (ev) CU_TRY(ctx, cudaEventRecord(ev[0], stream));
    if (n_pieces == 0) {
        if (int rc = launch_k1(ctx, walkers, n_walkers, false, stream)) return rc;
        if (ev) CU_TRY(ctx, cudaEventRecord(ev[1], stream));
        for (int s = 0; s < 2; ++s)
            if (ctx->sp[s].n > 0)
                if (int rc = launch_k2(ctx, s, 0, n_walkers, stream)) return rc;
    } else {
        for (int k = 0; k < n_pieces; ++k) {
            const EnergyPiece &pc = pieces[k];
            if (pc.wait) CU_TRY(ctx, cudaStreamWaitEvent(stream, pc.wait, 0));
            if (int rc = launch_k1(ctx, walkers, n_walkers, false, stream, pc.spin, pc.w0, pc.count)) return rc;
            if (ev && k == 0) CU_TRY(ctx, cudaEventRecord(ev[1], stream));
            if (int rc = launch_k2(ctx, pc.spin, pc.w0, pc.count, stream)) return rc;
        }
    }
    if (ev) CU_TRY(ctx, cudaEventRecord(ev[2], stream));

    // ---- K3 -------------------------------------------------------------------------------------------
    K3Params p3{};
    p3.n_gamma = ctx->n_gamma; p3.maxw = ctx->maxw; p3.e0 = ctx->e0;
    for (int s = 0; s < 2; ++s) {
        p3.n[s] = ctx->sp[s].n; p3.n_rt[s] = ctx->sp[s].n_rt; p3.tbuf[s] = ctx->sp[s].tbuf; p3.xpart[s] = ctx->sp[s].xpart;
    }
    p3.e1 = ctx->e1; p3.logdet = ctx->logdet;
    p3.out_energy = reinterpret_cast<double *>(out_energies);
    p3.out_overlap = reinterpret_cast<double *>(out_overlaps);
    k3_assemble<<<n_walkers, K3_THREADS, 0, stream>>>(p3);
    CU_TRY(ctx, cudaGetLastError());
    ctx->launches += 1;
    if (ev) { CU_TRY(ctx, cudaEventRecord(ev[3], stream)); ctx->prof_calls += 1; }
    ctx->last_nw = n_walkers;
    ctx->last_energy_nw = n_walkers;
    return AFQMC_OK;
}

int afqmc_local_energy(afqmc_ctx *ctx, const void *walkers, int n_walkers, void *out_energies, void *out_overlaps,
                       void *stream_) {
    if (!ctx) return AFQMC_ERR_ARG;
    if (!walkers || !out_energies || !out_overlaps) return fail(ctx, AFQMC_ERR_ARG, "afqmc_local_energy: null pointer argument");
    if (n_walkers < 1 || n_walkers > ctx->maxw)
        return fail(ctx, AFQMC_ERR_ARG, "afqmc_local_energy: n_walkers=%d outside 1..%d", n_walkers, ctx->maxw);
    return run_energy(ctx, walkers, n_walkers, out_energies, out_overlaps, (cudaStream_t)stream_, nullptr, 0);
}

int afqmc_local_energy_host(afqmc_ctx *ctx, const void *walkers_host, int n_walkers, void *out_energies_host,
                            void *out_overlaps_host, void *stream_) {
    if (!ctx) return AFQMC_ERR_ARG;
    if (!walkers_host || !out_energies_host || !out_overlaps_host)
        return fail(ctx, AFQMC_ERR_ARG, "afqmc_local_energy_host: null pointer argument");
    if (n_walkers < 1 || n_walkers > ctx->maxw)
        return fail(ctx, AFQMC_ERR_ARG, "afqmc_local_energy_host: n_walkers=%d outside 1..%d", n_walkers, ctx->maxw);
    cudaStream_t stream = (cudaStream_t)stream_;
    // Blocks of walkers are copied in the order the kernels want them: the first eighth of the first spin on `stream`,
    // then -- on the handle's copy stream, one event each -- the rest of that spin and the other spin.  K1 + K2 start on
    // the first block while the others land under them (K2 on an eighth of one spin takes several times longer than the
    // copy of everything that is left); only the first block's copy is exposed.
    const int N = ctx->N, na = ctx->sp[0].n, nb = ctx->sp[1].n;
    const char *src = reinterpret_cast<const char *>(walkers_host);
    char *dst = reinterpret_cast<char *>(ctx->h_walkers);
    const size_t a_bytes = (size_t)n_walkers * N * na * 16, b_bytes = (size_t)n_walkers * N * nb * 16;
    EnergyPiece pieces[3];
    int n_pieces = 0;
    const int s0 = na > 0 ? 0 : 1;                                        // first spin with electrons
    const size_t off0 = s0 == 0 ? 0 : a_bytes, row_bytes = (size_t)N * ctx->sp[s0].n * 16;
    const int wT = ctx->sp[s0].wT;
    int first = ((n_walkers + 7) / 8 + wT - 1) / wT * wT;               // an eighth, in whole K2 column tiles
    if (first >= n_walkers || n_walkers < 16 * wT) first = n_walkers;    // small batches: one block per spin
    CU_TRY(ctx, cudaMemcpyAsync(dst + off0, src + off0, first * row_bytes, cudaMemcpyHostToDevice, stream));
    CU_TRY(ctx, cudaEventRecord(ctx->ev_first, stream));                   // also orders the other copies after earlier work on `stream`
    CU_TRY(ctx, cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_first, 0));
    pieces[n_pieces++] = EnergyPiece{s0, 0, first, nullptr};
    if (first < n_walkers) {
        CU_TRY(ctx, cudaMemcpyAsync(dst + off0 + first * row_bytes, src + off0 + first * row_bytes, (n_walkers - first) * row_bytes,
                                    cudaMemcpyHostToDevice, ctx->copy_stream));
        CU_TRY(ctx, cudaEventRecord(ctx->ev_rest, ctx->copy_stream));
        pieces[n_pieces++] = EnergyPiece{s0, first, n_walkers - first, ctx->ev_rest};
    }
    if (s0 == 0 && nb > 0) {
        CU_TRY(ctx, cudaMemcpyAsync(dst + a_bytes, src + a_bytes, b_bytes, cudaMemcpyHostToDevice, ctx->copy_stream));
        CU_TRY(ctx, cudaEventRecord(ctx->ev_beta, ctx->copy_stream));
        pieces[n_pieces++] = EnergyPiece{1, 0, n_walkers, ctx->ev_beta};
    }
    if (int rc = run_energy(ctx, ctx->h_walkers, n_walkers, ctx->h_outE, ctx->h_outO, stream, pieces, n_pieces)) return rc;
    CU_TRY(ctx, cudaMemcpyAsync(out_energies_host, ctx->h_outE, (size_t)n_walkers * 16, cudaMemcpyDeviceToHost, stream));
    CU_TRY(ctx, cudaMemcpyAsync(out_overlaps_host, ctx->h_outO, (size_t)n_walkers * 16, cudaMemcpyDeviceToHost, stream));
    CU_TRY(ctx, cudaStreamSynchronize(stream));
    return AFQMC_OK;
}

int afqmc_force_bias(afqmc_ctx *ctx, void *out, void *stream_) {
    if (!ctx) return AFQMC_ERR_ARG;
    if (!out) return fail(ctx, AFQMC_ERR_ARG, "afqmc_force_bias: null pointer argument");
    if (ctx->last_energy_nw < 1) return fail(ctx, AFQMC_ERR_ARG, "afqmc_force_bias: no energy call has been made on this handle");
    const long long total = (long long)ctx->last_energy_nw * ctx->n_gamma * 2;
    k3_force_bias<<<(unsigned)((total + 255) / 256), 256, 0, (cudaStream_t)stream_>>>(
        ctx->last_energy_nw, ctx->n_gamma, ctx->sp[0].n, ctx->sp[1].n, ctx->sp[0].tbuf, ctx->sp[1].tbuf, reinterpret_cast<double *>(out));
    CU_TRY(ctx, cudaGetLastError());
    ctx->launches += 1;
    return AFQMC_OK;
}

int afqmc_enable_force_bias(afqmc_ctx *ctx, const double *chol, void *stream_) {
    if (!ctx) return AFQMC_ERR_ARG;
    if (!chol) return fail(ctx, AFQMC_ERR_ARG, "afqmc_enable_force_bias: null pointer argument");
    if (ctx->fb_enabled) return AFQMC_OK;
    cudaStream_t stream = (cudaStream_t)stream_;
    const int N = ctx->N, n_gamma = ctx->n_gamma, maxw = ctx->maxw;
    for (int s = 0; s < 2; ++s) {
        SpinCfg &sc = ctx->sp[s];
        const int n = sc.n;
        if (n == 0) continue;
        const int nbf = sc.cplx ? 2 : 1;                          // rows per gamma: Re (and Im) of Ltilde
        cudaFree(sc.f_A); cudaFree(sc.f_B); cudaFree(sc.f_craw);  // a failed earlier attempt may have left some behind
        sc.f_A = sc.f_B = sc.f_craw = nullptr;
        sc.f_wT = std::min(64, (maxw + 3) / 4 * 4);               // 2 * wT columns = 8 * NT
        sc.f_NT = sc.f_wT / 4;
        sc.f_strips = std::min(K2_MAX_WM, (n_gamma * nbf + 7) / 8);
        sc.f_gT = sc.f_strips * 8 / nbf;
        sc.f_n_rt = (n_gamma + sc.f_gT - 1) / sc.f_gT;
        sc.f_n_ct_max = (maxw + sc.f_wT - 1) / sc.f_wT;
        // split K so that (row tiles x column tiles x K parts) fills whole rounds of the persistent grid
        const int ks_raw = (n * N + 3) / 4;
        sc.f_ksc = std::min(12, ks_raw);
        int best_s = 1;
        double best_fill = 0.0;
        for (int sp = 1; sp <= 8; ++sp) {
            if (ks_raw / sp < 4 * sc.f_ksc && sp > 1) break;     // keep every part at least a few chunks long
            const long long items = (long long)sc.f_n_rt * sc.f_n_ct_max * sp;
            const long long rounds = (items + ctx->num_sms - 1) / ctx->num_sms;
            const double fill = (double)items / (double)(rounds * ctx->num_sms);
            if (fill > best_fill + 0.02) { best_fill = fill; best_s = sp; }
        }
        sc.f_ksplit = best_s;
        sc.f_kps = ((ks_raw + best_s - 1) / best_s + sc.f_ksc - 1) / sc.f_ksc * sc.f_ksc;   // k-steps per part, whole chunks
        sc.f_ksteps = sc.f_kps * best_s;                                                   // padded with zero k-steps
        sc.f_nchunks = sc.f_kps / sc.f_ksc;
        sc.f_nstages = 2;
        sc.f_smem = (size_t)sc.f_nstages * sc.f_ksc * (sc.f_strips + sc.f_NT) * 256 + (size_t)2 * sc.f_nstages * 8 + 16;
        sc.f_layA = OperandLayout{1, sc.f_strips, sc.f_ksteps, sc.f_gT, (long long)sc.f_strips * sc.f_ksteps * 32};
        sc.f_layB = OperandLayout{1, sc.f_NT, sc.f_ksteps, sc.f_wT, (long long)sc.f_NT * sc.f_ksteps * 32};
        const size_t a_bytes = (size_t)sc.f_n_rt * sc.f_layA.tile_doubles * 8, b_bytes = (size_t)sc.f_n_ct_max * sc.f_layB.tile_doubles * 8;
        const size_t c_bytes = (size_t)sc.f_ksplit * n_gamma * nbf * sc.f_n_ct_max * sc.f_NT * 8 * 8;
        CU_TRY(ctx, cudaMalloc(&sc.f_A, a_bytes));
        CU_TRY(ctx, cudaMalloc(&sc.f_B, b_bytes));
        CU_TRY(ctx, cudaMalloc(&sc.f_craw, c_bytes));
        CU_TRY(ctx, cudaMemsetAsync(sc.f_A, 0, a_bytes, stream));
        CU_TRY(ctx, cudaMemsetAsync(sc.f_B, 0, b_bytes, stream));
        dim3 grid(n_gamma, (N + 127) / 128);
        k0_half_rotate_chol<<<grid, 128, 0, stream>>>(chol, sc.psi, N, n, n_gamma, n * nbf, 0, 1.0, OperandLayout{}, nullptr, sc.f_layA, sc.f_A);
        CU_TRY(ctx, cudaGetLastError());
        ctx->launches += 1;
        if (sc.cplx) {
            k0_half_rotate_chol<<<grid, 128, 0, stream>>>(chol, sc.psi_im, N, n, n_gamma, n * nbf, n, -1.0, OperandLayout{}, nullptr, sc.f_layA, sc.f_A);
            CU_TRY(ctx, cudaGetLastError());
            ctx->launches += 1;
        }
        K2FbFn fn = k2_pick_fb(sc.f_NT);
        if (!fn) return fail(ctx, AFQMC_ERR_UNSUPPORTED, "afqmc_enable_force_bias: no kernel for NT=%d", sc.f_NT);
        CU_TRY(ctx, allow_max_smem(fn));
    }
    CU_TRY(ctx, cudaStreamSynchronize(stream));
    ctx->fb_enabled = true;
    return AFQMC_OK;
}

int afqmc_force_bias_only(afqmc_ctx *ctx, const void *walkers, int n_walkers, void *out, void *stream_) {
    if (!ctx) return AFQMC_ERR_ARG;
    if (!walkers || !out) return fail(ctx, AFQMC_ERR_ARG, "afqmc_force_bias_only: null pointer argument");
    if (!ctx->fb_enabled) return fail(ctx, AFQMC_ERR_ARG, "afqmc_force_bias_only: call afqmc_enable_force_bias first");
    if (n_walkers < 1 || n_walkers > ctx->maxw)
        return fail(ctx, AFQMC_ERR_ARG, "afqmc_force_bias_only: n_walkers=%d outside 1..%d", n_walkers, ctx->maxw);
    cudaStream_t stream = (cudaStream_t)stream_;
    if (int rc = launch_k1(ctx, walkers, n_walkers, true, stream)) return rc;
    if (int rc = launch_force_bias_gemm(ctx, n_walkers, reinterpret_cast<double *>(out), stream)) return rc;
    ctx->last_nw = n_walkers;
    return AFQMC_OK;
}

int afqmc_spin_squared(afqmc_ctx *ctx, void *out, void *stream_) {
    if (!ctx) return AFQMC_ERR_ARG;
    if (!out) return fail(ctx, AFQMC_ERR_ARG, "afqmc_spin_squared: null pointer argument");
    if (ctx->last_nw < 1) return fail(ctx, AFQMC_ERR_ARG, "afqmc_spin_squared: no energy or force-bias call has been made on this handle");
    K5Params p5{};
    p5.N = ctx->N; p5.n_walkers = ctx->last_nw; p5.out = reinterpret_cast<double *>(out);
    for (int s = 0; s < 2; ++s) {
        p5.n[s] = ctx->sp[s].n; p5.theta[s] = ctx->sp[s].B; p5.layB[s] = ctx->sp[s].layB;
        p5.psi[s] = ctx->sp[s].psi; p5.psi_im[s] = ctx->sp[s].psi_im;
    }
    const int na = p5.n[0], nb = p5.n[1];
    const size_t smem = ((size_t)2 * na * nb + (size_t)2 * (na + nb) * K5_PCHUNK) * 16;
    k5_spin_squared<<<ctx->last_nw, K5_THREADS, smem, (cudaStream_t)stream_>>>(p5);
    CU_TRY(ctx, cudaGetLastError());
    ctx->launches += 1;
    return AFQMC_OK;
}

int afqmc_greens_function(afqmc_ctx *ctx, int spin, void *out, void *stream_) {
    if (!ctx) return AFQMC_ERR_ARG;
    if (!out || (spin != 0 && spin != 1)) return fail(ctx, AFQMC_ERR_ARG, "afqmc_greens_function: bad argument");
    if (ctx->last_nw < 1) return fail(ctx, AFQMC_ERR_ARG, "afqmc_greens_function: no energy or force-bias call has been made on this handle");
    const SpinCfg &sc = ctx->sp[spin];
    const int N = ctx->N;
    if (sc.n == 0) {        // empty spin sector: G = 0
        CU_TRY(ctx, cudaMemsetAsync(out, 0, (size_t)ctx->last_nw * N * N * 16, (cudaStream_t)stream_));
        return AFQMC_OK;
    }
    K6Params p6{};
    p6.N = N; p6.n = sc.n; p6.theta = sc.B; p6.layB = sc.layB; p6.psi = sc.psi; p6.psi_im = sc.psi_im;
    p6.out = reinterpret_cast<double2 *>(out);
    const size_t smem = (size_t)2 * sc.n * K6_TILE * 16;
    const int nt = (N + K6_TILE - 1) / K6_TILE;
    k6_greens_function<<<dim3(ctx->last_nw, nt, nt), 256, smem, (cudaStream_t)stream_>>>(p6);
    CU_TRY(ctx, cudaGetLastError());
    ctx->launches += 1;
    return AFQMC_OK;
}

int afqmc_phaseless_weights(int n_walkers, int n_gamma, const double *x, const void *xbar, const void *log_ovlp_old,
                            const void *log_ovlp_new, const double *weights_in, double *weights_out, void *stream_) {
    if (n_walkers < 1 || n_gamma < 1 || !x || !xbar || !log_ovlp_old || !log_ovlp_new || !weights_in || !weights_out)
        return fail(nullptr, AFQMC_ERR_ARG, "afqmc_phaseless_weights: bad argument");
    k7_phaseless_update<<<n_walkers, K7_THREADS, 0, (cudaStream_t)stream_>>>(
        n_gamma, x, reinterpret_cast<const double *>(xbar), reinterpret_cast<const double *>(log_ovlp_old),
        reinterpret_cast<const double *>(log_ovlp_new), weights_in, weights_out);
    CU_TRY(nullptr, cudaGetLastError());
    return AFQMC_OK;
}

int afqmc_sample_fields(unsigned long long seed, unsigned long long step, int first_walker, int n_walkers, int n_gamma, double *x,
                        void *stream_) {
    if (n_walkers < 1 || n_gamma < 1 || first_walker < 0 || !x) return fail(nullptr, AFQMC_ERR_ARG, "afqmc_sample_fields: bad argument");
    const long long pairs = (long long)n_walkers * ((n_gamma + 1) / 2);
    k10_sample_fields<<<(unsigned)((pairs + 255) / 256), 256, 0, (cudaStream_t)stream_>>>(seed, step, first_walker, n_walkers, n_gamma, x);
    CU_TRY(nullptr, cudaGetLastError());
    return AFQMC_OK;
}

int afqmc_enable_propagation(afqmc_ctx *ctx, const double *h1e, const double *chol, double dt, void *stream_) {
    if (!ctx) return AFQMC_ERR_ARG;
    if (!h1e || !chol) return fail(ctx, AFQMC_ERR_ARG, "afqmc_enable_propagation: null pointer argument");
    if (!(dt > 0.0) || !std::isfinite(dt)) return fail(ctx, AFQMC_ERR_ARG, "afqmc_enable_propagation: dt must be positive and finite");
    if (ctx->prop_enabled) return fail(ctx, AFQMC_ERR_ARG, "afqmc_enable_propagation: already enabled on this handle (dt = %g)", ctx->dt);
    cudaStream_t stream = (cudaStream_t)stream_;
    if (int rc = afqmc_enable_force_bias(ctx, chol, stream_)) return rc;
    const int N = ctx->N, n_gamma = ctx->n_gamma, maxw = ctx->maxw;
    const int C = 2 * (ctx->sp[0].n + ctx->sp[1].n);
    ctx->dt = dt;
    ctx->ldE = (N + 1) & ~1; ctx->ldt = C;                        // even pitches: K9 stores (re, im) pairs as double2
    const int S = (N + 7) / 8;
    ctx->p_row_tiles = (S + K9_MAXROWS / 8 - 1) / (K9_MAXROWS / 8);
    ctx->p_rt_strips = (S + ctx->p_row_tiles - 1) / ctx->p_row_tiles;
    CU_TRY(ctx, allow_max_smem(k9_apply));
    CU_TRY(ctx, allow_max_smem(k2_force_bias<16>));

    // ---- h' = h - 1/2 sum_g (L^g)^2 and E = exp(-dt h'/2) by scaling and squaring (all products in K9) -------------
    const size_t ebytes = (size_t)N * ctx->ldE * 8;
    CU_TRY(ctx, cudaMalloc(&ctx->hp, (size_t)N * N * 8));
    CU_TRY(ctx, cudaMalloc(&ctx->Emat, ebytes));
    CU_TRY(ctx, cudaMalloc(&ctx->Etmp[0], ebytes));
    CU_TRY(ctx, cudaMalloc(&ctx->Etmp[1], ebytes));
    k8_one_body_shift<<<dim3((N + 15) / 16, (N + 15) / 16), 256, 0, stream>>>(h1e, chol, N, n_gamma, ctx->hp);
    CU_TRY(ctx, cudaGetLastError());
    std::vector<double> hp_h((size_t)N * N);
    CU_TRY(ctx, cudaMemcpyAsync(hp_h.data(), ctx->hp, hp_h.size() * 8, cudaMemcpyDeviceToHost, stream));
    CU_TRY(ctx, cudaStreamSynchronize(stream));
    double norm1 = 0.0;                                           // picks the number of squarings only
    for (int q = 0; q < N; ++q) {
        double c = 0.0;
        for (int p = 0; p < N; ++p) c += std::fabs(hp_h[(size_t)p * N + q]);
        norm1 = std::max(norm1, c);
    }
    if (!std::isfinite(norm1)) return fail(ctx, AFQMC_ERR_ARG, "afqmc_enable_propagation: h1e / chol have non-finite entries");
    int nsq = 0;
    while (0.5 * dt * norm1 / std::ldexp(1.0, nsq) > 0.5 && nsq < 60) ++nsq;
    double *term = ctx->Etmp[0], *next = ctx->Etmp[1], *sum = ctx->Emat;
    CU_TRY(ctx, cudaMemsetAsync(term, 0, ebytes, stream));
    CU_TRY(ctx, cudaMemsetAsync(next, 0, ebytes, stream));
    CU_TRY(ctx, cudaMemsetAsync(sum, 0, ebytes, stream));
    k8_set_diagonal<<<(N + 255) / 256, 256, 0, stream>>>(term, N, ctx->ldE, 1.0);
    k8_set_diagonal<<<(N + 255) / 256, 256, 0, stream>>>(sum, N, ctx->ldE, 1.0);
    CU_TRY(ctx, cudaGetLastError());
    for (int k = 1; k <= 18; ++k) {                               // ||X|| <= 1/2: the 18th term is below 1e-21
        const double alpha = -0.5 * dt / std::ldexp(1.0, nsq) / k;
        if (int rc = launch_k9(ctx, ctx->hp, nullptr, 0, N, term, next, sum, 0, ctx->ldE, N, 1, alpha, stream)) return rc;
        std::swap(term, next);
    }
    double *cur = sum, *other = term;                             // `term` and `next` are free now
    for (int k = 0; k < nsq; ++k) {
        if (int rc = launch_k9(ctx, cur, nullptr, 0, ctx->ldE, cur, other, nullptr, 0, ctx->ldE, N, 1, 1.0, stream)) return rc;
        std::swap(cur, other);
    }
    if (cur != ctx->Emat) CU_TRY(ctx, cudaMemcpyAsync(ctx->Emat, cur, ebytes, cudaMemcpyDeviceToDevice, stream));

    // ---- operands of the field GEMM  A(y)_w[pq] = sum_g c_wg L^g[pq] ------------------------------------------------
    const int ksteps = (n_gamma + 3) / 4;
    ctx->v_ksc = std::min(12, ksteps);
    ctx->v_kps = (ksteps + ctx->v_ksc - 1) / ctx->v_ksc * ctx->v_ksc;
    ctx->v_nchunks = ctx->v_kps / ctx->v_ksc;
    ctx->v_nstages = 2;
    // Rows of the GEMM are the pairs p <= q (upper triangle: L^g and A(y) are symmetric), 96 per tile, so that the big
    // operand -- the Cholesky vectors, 8 Ngamma N (N + 1) / 2 bytes -- streams from HBM exactly once and every warp of
    // the CTA owns a strip; columns are (walker, re / im) of the coefficients, 128 per tile.
    const long long npq = (long long)N * (N + 1) / 2;
    ctx->v_strips = K2_MAX_WM;
    const int rtiles = (int)((npq + 8 * ctx->v_strips - 1) / (8 * ctx->v_strips));
    ctx->v_n_ct = (2 * maxw + 127) / 128;
    ctx->ldv = (long long)ctx->v_n_ct * 128;
    ctx->v_smem = (size_t)ctx->v_nstages * ctx->v_ksc * (ctx->v_strips + 16) * 256 + (size_t)2 * ctx->v_nstages * 8 + 16;
    ctx->v_layA = OperandLayout{1, ctx->v_strips, ctx->v_kps, ctx->v_strips * 8, (long long)ctx->v_strips * ctx->v_kps * 32};
    ctx->v_layB = OperandLayout{1, 16, ctx->v_kps, 128, (long long)16 * ctx->v_kps * 32};
    const size_t a_bytes = (size_t)rtiles * ctx->v_layA.tile_doubles * 8, b_bytes = (size_t)ctx->v_n_ct * ctx->v_layB.tile_doubles * 8;
    CU_TRY(ctx, cudaMalloc(&ctx->v_A, a_bytes));
    CU_TRY(ctx, cudaMalloc(&ctx->v_B, b_bytes));
    CU_TRY(ctx, cudaMemsetAsync(ctx->v_A, 0, a_bytes, stream));
    CU_TRY(ctx, cudaMemsetAsync(ctx->v_B, 0, b_bytes, stream));
    if (ksteps > 65535 || N > 65535) return fail(ctx, AFQMC_ERR_UNSUPPORTED, "afqmc_enable_propagation: n_gamma > 262140 or N > 65535 is not supported");
    k8_pack_chol_vhs<<<dim3((N + 127) / 128, N, ksteps), 128, 0, stream>>>(chol, N, n_gamma, ctx->v_layA, ctx->v_A);
    CU_TRY(ctx, cudaGetLastError());
    ctx->launches += 4 + 18 + nsq;

    // ---- work buffers ------------------------------------------------------------------------------------------------
    CU_TRY(ctx, cudaMalloc(&ctx->Vtri, (size_t)rtiles * 8 * ctx->v_strips * ctx->ldv * 8));      // [pair p <= q][(walker, re / im)]
    CU_TRY(ctx, cudaMalloc(&ctx->V, (size_t)2 * maxw * N * N * 8));
    CU_TRY(ctx, cudaMalloc(&ctx->fbuf, (size_t)maxw * n_gamma * 16));
    CU_TRY(ctx, cudaMalloc(&ctx->xbar, (size_t)maxw * n_gamma * 16));
    for (int k = 0; k < 3; ++k) CU_TRY(ctx, cudaMalloc(&ctx->Tb[k], (size_t)maxw * N * ctx->ldt * 8));
    CU_TRY(ctx, cudaMalloc(&ctx->lo_old, (size_t)maxw * 16));
    CU_TRY(ctx, cudaMalloc(&ctx->lo_new, (size_t)maxw * 16));
    for (auto &e : ctx->pev) CU_TRY(ctx, cudaEventCreate(&e));
    CU_TRY(ctx, cudaStreamSynchronize(stream));
    ctx->prop_enabled = true;
    return AFQMC_OK;
}

int afqmc_propagate(afqmc_ctx *ctx, void *walkers, int n_walkers, const double *x, const double *weights_in,
                    double *weights_out, void *log_ovlp_out, int taylor_order, void *stream_) {
    if (!ctx) return AFQMC_ERR_ARG;
    if (!walkers || !x || !weights_in || !weights_out) return fail(ctx, AFQMC_ERR_ARG, "afqmc_propagate: null pointer argument");
    if (!ctx->prop_enabled) return fail(ctx, AFQMC_ERR_ARG, "afqmc_propagate: call afqmc_enable_propagation first");
    if (n_walkers < 1 || n_walkers > ctx->maxw)
        return fail(ctx, AFQMC_ERR_ARG, "afqmc_propagate: n_walkers=%d outside 1..%d", n_walkers, ctx->maxw);
    if (taylor_order < 0 || taylor_order > 64) return fail(ctx, AFQMC_ERR_ARG, "afqmc_propagate: taylor_order=%d outside 0..64", taylor_order);
    cudaStream_t stream = (cudaStream_t)stream_;
    const int N = ctx->N, n_gamma = ctx->n_gamma, na = ctx->sp[0].n, nb = ctx->sp[1].n, C = 2 * (na + nb), ld = ctx->ldt;
    const long long tstride = (long long)N * ld;
    cudaEvent_t *ev = ctx->profiling ? ctx->pev : nullptr;
    int evi = 0;
    auto mark = [&]() -> cudaError_t { return ev ? cudaEventRecord(ev[evi++], stream) : cudaSuccess; };
    CU_TRY(ctx, mark());

    // (1) theta, log-overlap of phi (Eq. 16, 23) and the force bias sum_pq G_pq L^g_pq (Eq. 19 / 24)
    if (int rc = launch_k1(ctx, walkers, n_walkers, true, stream)) return rc;
    k8_log_overlap<<<(n_walkers + 127) / 128, 128, 0, stream>>>(n_walkers, ctx->maxw, na, nb, ctx->logdet, ctx->lo_old);
    CU_TRY(ctx, cudaGetLastError());
    CU_TRY(ctx, mark());
    if (int rc = launch_force_bias_gemm(ctx, n_walkers, ctx->fbuf, stream)) return rc;
    CU_TRY(ctx, mark());

    // (2) xbar (Eq. 9) and the coefficients of A(x - xbar); A(y)_w = sum_g c_wg L^g on the FP64 tensor cores
    const long long nf = (long long)n_walkers * ((n_gamma + 3) / 4);
    k8_fields<<<(unsigned)((nf + 255) / 256), 256, 0, stream>>>(n_walkers, n_gamma, ctx->dt, ctx->fbuf, x, ctx->xbar, ctx->v_layB, ctx->v_B);
    CU_TRY(ctx, cudaGetLastError());
    {
        K2FbParams p2{};
        p2.A = ctx->v_A; p2.B = ctx->v_B;
        p2.itemA_doubles = ctx->v_layA.tile_doubles; p2.tileB_doubles = ctx->v_layB.tile_doubles; p2.partB_doubles = 0;
        const long long npq = (long long)N * (N + 1) / 2;
        p2.rows_per_tile = ctx->v_strips * 8; p2.rows_total = (int)npq;
        p2.strips = ctx->v_strips; p2.WM = K2_MAX_WM;
        p2.kps = ctx->v_kps; p2.ksc = ctx->v_ksc; p2.nchunks = ctx->v_nchunks; p2.nstages = ctx->v_nstages;
        p2.n_items_r = (int)((npq + p2.rows_per_tile - 1) / p2.rows_per_tile); p2.ksplit = 1; p2.n_ct = (2 * n_walkers + 127) / 128;
        p2.craw = ctx->Vtri;
        const long long ntiles = (long long)p2.n_items_r * p2.n_ct;
        k2_force_bias<16><<<(int)std::min<long long>(ntiles, ctx->num_sms), 32 * K2_MAX_WM, ctx->v_smem, stream>>>(p2);
        CU_TRY(ctx, cudaGetLastError());
        if (N > 65535) return fail(ctx, AFQMC_ERR_UNSUPPORTED, "afqmc_propagate: N > 65535");
        k8_expand_symmetric<<<dim3((N + 31) / 32, N, (2 * n_walkers + 31) / 32), dim3(32, 8), 0, stream>>>(
            ctx->Vtri, (long long)p2.n_ct * 128, N, 2 * n_walkers, ctx->V);
        CU_TRY(ctx, cudaGetLastError());
    }
    CU_TRY(ctx, mark());

    // (3) phi' = E exp(A) E phi (Eq. 13): T0 = E phi, S = sum_k A^k T0 / k!, phi' = E S
    double *X0 = ctx->Tb[0], *X1 = ctx->Tb[1], *X2 = ctx->Tb[2];
    const long long np = (long long)n_walkers * N * ld;
    k8_pack_walkers<<<(unsigned)((np + 255) / 256), 256, 0, stream>>>(reinterpret_cast<const double *>(walkers), n_walkers, N, na, nb, ld, X0);
    CU_TRY(ctx, cudaGetLastError());
    if (int rc = launch_k9(ctx, ctx->Emat, nullptr, 0, ctx->ldE, X0, X1, nullptr, tstride, ld, C, n_walkers, 1.0, stream)) return rc;   // T0 = E phi
    // sum_{k <= order} A^k T0 / k!  by Horner's rule:  R_order = T0,  R_{j-1} = T0 + A R_j / j,  result R_0  (the same
    // polynomial as the term-by-term sum; one read of T0 per step instead of a read-modify-write of a running sum)
    const double *R = X1;
    double *bufs[2] = {X0, X2};
    for (int j = taylor_order; j >= 1; --j) {
        double *out = bufs[(taylor_order - j) & 1];
        if (int rc = launch_k9(ctx, ctx->V, ctx->V + (long long)N * N, 2LL * N * N, N, R, out, nullptr, tstride, ld, C, n_walkers, 1.0 / j, stream, X1)) return rc;
        R = out;
    }
    double *cur = (R == X0) ? X2 : X0;                            // any buffer other than R (X1 is free after the last step too)
    if (int rc = launch_k9(ctx, ctx->Emat, nullptr, 0, ctx->ldE, R, cur, nullptr, tstride, ld, C, n_walkers, 1.0, stream)) return rc;
    const long long nu = (long long)n_walkers * N * C;
    k8_unpack_walkers<<<(unsigned)((nu + 255) / 256), 256, 0, stream>>>(cur, n_walkers, N, na, nb, ld, reinterpret_cast<double *>(walkers));
    CU_TRY(ctx, cudaGetLastError());
    CU_TRY(ctx, mark());

    // (4) overlap of phi' (Eq. 8) and the phaseless weights (Eq. 7, 10-12)
    if (int rc = launch_k1(ctx, walkers, n_walkers, false, stream)) return rc;
    k8_log_overlap<<<(n_walkers + 127) / 128, 128, 0, stream>>>(n_walkers, ctx->maxw, na, nb, ctx->logdet, ctx->lo_new);
    CU_TRY(ctx, cudaGetLastError());
    k7_phaseless_update<<<n_walkers, K7_THREADS, 0, stream>>>(n_gamma, x, ctx->xbar, ctx->lo_old, ctx->lo_new, weights_in, weights_out);
    CU_TRY(ctx, cudaGetLastError());
    if (log_ovlp_out) CU_TRY(ctx, cudaMemcpyAsync(log_ovlp_out, ctx->lo_new, (size_t)n_walkers * 16, cudaMemcpyDeviceToDevice, stream));
    CU_TRY(ctx, mark());
    ctx->pev_valid = ev != nullptr;
    ctx->launches += 10 + taylor_order;
    ctx->last_nw = n_walkers;
    ctx->last_energy_nw = 0;            // the Coulomb traces in the handle belong to other walkers now
    return AFQMC_OK;
}

int afqmc_propagate_phase_ms(afqmc_ctx *ctx, float ms[5]) {
    if (!ctx || !ms) return AFQMC_ERR_ARG;
    if (!ctx->pev_valid) return fail(ctx, AFQMC_ERR_ARG, "afqmc_propagate_phase_ms: no profiled afqmc_propagate call recorded");
    for (int k = 0; k < 5; ++k) CU_TRY(ctx, cudaEventElapsedTime(&ms[k], ctx->pev[k], ctx->pev[k + 1]));
    return AFQMC_OK;
}

int afqmc_propagation_xbar(afqmc_ctx *ctx, void *out, void *stream_) {
    if (!ctx) return AFQMC_ERR_ARG;
    if (!out) return fail(ctx, AFQMC_ERR_ARG, "afqmc_propagation_xbar: null pointer argument");
    if (!ctx->prop_enabled || ctx->last_nw < 1) return fail(ctx, AFQMC_ERR_ARG, "afqmc_propagation_xbar: no afqmc_propagate call has been made");
    CU_TRY(ctx, cudaMemcpyAsync(out, ctx->xbar, (size_t)ctx->last_nw * ctx->n_gamma * 16, cudaMemcpyDeviceToDevice, (cudaStream_t)stream_));
    return AFQMC_OK;
}

void afqmc_destroy(afqmc_ctx *ctx) { free_ctx(ctx); }

const char *afqmc_last_error(const afqmc_ctx *ctx) { return ctx ? ctx->err.c_str() : g_create_error.c_str(); }

static void fill_info(afqmc_info *info, int N, int n_gamma, int maxw, const SpinCfg sp[2]) {
    std::memset(info, 0, sizeof *info);
    info->N = N; info->n_alpha = sp[0].n; info->n_beta = sp[1].n; info->n_gamma = n_gamma;
    info->max_walkers = maxw; info->k_steps = (N + 3) / 4;
    for (int s = 0; s < 2; ++s) {
        const SpinCfg &c = sp[s];
        info->tile_rows[s] = c.strips * 8; info->tile_cols[s] = c.NT * 8;
        info->gammas_per_tile[s] = c.gT; info->walkers_per_tile[s] = c.wT;
        info->warps_m[s] = c.WM; info->mt[s] = c.MT; info->nt[s] = c.NT; info->stages[s] = c.nstages;
        info->ksteps_per_chunk[s] = c.ksc; info->k2_smem_bytes[s] = (int)c.k2_smem;
        info->ltilde_bytes += (long long)c.A_bytes; info->theta_bytes += (long long)c.B_bytes;
    }
}

int afqmc_get_info(const afqmc_ctx *ctx, afqmc_info *info) {
    if (!ctx || !info) return AFQMC_ERR_ARG;
    fill_info(info, ctx->N, ctx->n_gamma, ctx->maxw, ctx->sp);
    info->kernel_launches = ctx->launches;
    return AFQMC_OK;
}

int afqmc_plan(int N, int n_alpha, int n_beta, int n_gamma, int max_walkers, afqmc_info *info) {
    return afqmc_plan_trial(N, n_alpha, n_beta, n_gamma, max_walkers, 0, 0, info);
}

int afqmc_plan_trial(int N, int n_alpha, int n_beta, int n_gamma, int max_walkers, int complex_alpha, int complex_beta,
                     afqmc_info *info) {
    if (!info) return fail(nullptr, AFQMC_ERR_ARG, "afqmc_plan: null pointer argument");
    if (N < 1 || n_gamma < 1 || max_walkers < 1 || n_alpha < 0 || n_beta < 0 || n_alpha > N || n_beta > N ||
        n_alpha + n_beta < 1)
        return fail(nullptr, AFQMC_ERR_ARG, "afqmc_plan: size out of range");
    if (n_alpha > AFQMC_MAX_NOCC || n_beta > AFQMC_MAX_NOCC)
        return fail(nullptr, AFQMC_ERR_UNSUPPORTED, "afqmc_plan: n_sigma > %d is not supported yet", AFQMC_MAX_NOCC);
    SpinCfg sp[2];
    const int ns[2] = {n_alpha, n_beta};
    const bool cx[2] = {complex_alpha != 0, complex_beta != 0};
    for (int s = 0; s < 2; ++s)
        if (!choose_cfg(ns[s], cx[s], N, n_gamma, max_walkers, sp[s]))
            return fail(nullptr, AFQMC_ERR_UNSUPPORTED, "afqmc_plan: no K2 tile shape fits n_sigma=%d", ns[s]);
    fill_info(info, N, n_gamma, max_walkers, sp);
    return AFQMC_OK;
}

int afqmc_set_profiling(afqmc_ctx *ctx, int enable) {
    if (!ctx) return AFQMC_ERR_ARG;
    if (enable && ctx->ev.empty()) {
        ctx->ev.assign((size_t)kProfSets * 4, nullptr);
        for (auto &e : ctx->ev) CU_TRY(ctx, cudaEventCreate(&e));
    }
    ctx->profiling = enable != 0;
    ctx->prof_calls = 0;
    return AFQMC_OK;
}

int afqmc_last_kernel_ms(afqmc_ctx *ctx, float ms[3]) {
    if (!ctx || !ms) return AFQMC_ERR_ARG;
    if (ctx->prof_calls < 1) return fail(ctx, AFQMC_ERR_ARG, "afqmc_last_kernel_ms: no profiled call recorded");
    const cudaEvent_t *ev = &ctx->ev[(size_t)((ctx->prof_calls - 1) % kProfSets) * 4];
    for (int k = 0; k < 3; ++k) CU_TRY(ctx, cudaEventElapsedTime(&ms[k], ev[k], ev[k + 1]));
    return AFQMC_OK;
}

int afqmc_mean_kernel_ms(afqmc_ctx *ctx, float ms[3], int *n_calls) {
    if (!ctx || !ms || !n_calls) return AFQMC_ERR_ARG;
    if (ctx->prof_calls < 1) return fail(ctx, AFQMC_ERR_ARG, "afqmc_mean_kernel_ms: no profiled call recorded");
    const int cnt = (int)std::min<long long>(ctx->prof_calls, kProfSets);
    double acc[3] = {0.0, 0.0, 0.0};
    for (int c = 0; c < cnt; ++c) {
        const cudaEvent_t *ev = &ctx->ev[(size_t)c * 4];
        for (int k = 0; k < 3; ++k) {
            float t = 0.f;
            CU_TRY(ctx, cudaEventElapsedTime(&t, ev[k], ev[k + 1]));
            acc[k] += t;
        }
    }
    for (int k = 0; k < 3; ++k) ms[k] = (float)(acc[k] / cnt);
    *n_calls = cnt;
    return AFQMC_OK;
}

int afqmc_fp64_peak(int mode, int launches, double *tflops, void *stream_) {
    if (!tflops || launches < 1 || (mode != 0 && mode != 1)) return fail(nullptr, AFQMC_ERR_ARG, "afqmc_fp64_peak: bad argument");
    int sms = 0;
    if (int rc = check_arch(nullptr, &sms)) return rc;
    cudaStream_t stream = (cudaStream_t)stream_;
    double *d = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    struct Cleanup {                                   // releases the scratch on every return path
        double *&d; cudaEvent_t &e0, &e1;
        ~Cleanup() { if (e0) cudaEventDestroy(e0); if (e1) cudaEventDestroy(e1); cudaFree(d); }
    } cleanup{d, e0, e1};
    CU_TRY(nullptr, cudaMalloc(&d, 8));
    CU_TRY(nullptr, cudaEventCreate(&e0));
    CU_TRY(nullptr, cudaEventCreate(&e1));
    const int iters = mode == 0 ? 20000 : 50000;
    const int threads = 512;
    auto launch = [&]() {
        if (mode == 0) peak_dmma<<<sms, threads, 0, stream>>>(d, iters, 1.0000001, 1e-9);
        else peak_dfma<<<2 * sms, threads, 0, stream>>>(d, iters, 1.0000001, 1e-9);
    };
    launch();
    CU_TRY(nullptr, cudaStreamSynchronize(stream));
    CU_TRY(nullptr, cudaEventRecord(e0, stream));
    for (int k = 0; k < launches; ++k) launch();
    CU_TRY(nullptr, cudaEventRecord(e1, stream));
    CU_TRY(nullptr, cudaEventSynchronize(e1));
    float ms = 0.f;
    CU_TRY(nullptr, cudaEventElapsedTime(&ms, e0, e1));
    const double flops = mode == 0 ? 2.0 * 256 * PEAK_NACC * (double)iters * (threads / 32) * sms * launches
                                   : 2.0 * PEAK_NCH * (double)iters * threads * 2 * sms * launches;
    *tflops = flops / (ms * 1e-3) * 1e-12;
    return AFQMC_OK;
}

#ifdef AFQMC_K1_PHASE_CLOCKS
// Diagnostic builds only (k1_overlap.cuh): out[0] = K1 CTAs run since the last call, out[1..7] = cycles from CTA start
// to each phase boundary, summed over those CTAs.  Resets the counters.
int afqmc_k1_phase_clocks(long long out[8]) {
    if (!out) return AFQMC_ERR_ARG;
    CU_TRY(nullptr, cudaDeviceSynchronize());
    CU_TRY(nullptr, cudaMemcpyFromSymbol(out, afqmc::g_k1_clocks, 8 * sizeof(long long)));
    const long long zero[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    CU_TRY(nullptr, cudaMemcpyToSymbol(afqmc::g_k1_clocks, zero, sizeof zero));
    return AFQMC_OK;
}
#endif

}  // extern "C"

// ---- afqmc_log_overlap_static: an entry point that allocates nothing ------------------------------------------------------
// Its scratch (psi^T fragment planes, a zero block standing in for htilde, the packed theta K1 writes, K1's per-walker
// outputs) lives in this file-scope array: every GPU that loads the library holds AFQMC_STATIC_SCRATCH_BYTES of it until
// the process exits.  In host code the array's name is only a host-side stand-in; the device address comes from
// cudaGetSymbolAddress, once per device (static_scratch_for_current_device).
static __device__ __align__(256) unsigned char g_static_scratch[AFQMC_STATIC_SCRATCH_BYTES];

namespace {

constexpr int kMaxDevices = 64;
std::mutex g_static_mutex;
unsigned char *g_static_ptr[kMaxDevices] = {};

// Device address of g_static_scratch on the current device; first use on a device also opts the K1 kernels in to their
// dynamic shared memory there.  No allocation.
int static_scratch_for_current_device(unsigned char **out) {
    int dev = 0;
    CU_TRY(nullptr, cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return fail(nullptr, AFQMC_ERR_UNSUPPORTED, "afqmc_log_overlap_static: device ordinal %d >= %d", dev, kMaxDevices);
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[dev]) {
        unsigned char *ptr = nullptr;
        CU_TRY(nullptr, cudaGetSymbolAddress((void **)&ptr, g_static_scratch));
        if (!ptr) return fail(nullptr, AFQMC_ERR_CUDA, "afqmc_log_overlap_static: cudaGetSymbolAddress returned a null address");
        CU_TRY(nullptr, allow_max_smem(k1_overlap_inverse_theta<0, false>));
        CU_TRY(nullptr, allow_max_smem(k1_overlap_inverse_theta<1, false>));
        CU_TRY(nullptr, allow_max_smem(k1_overlap_inverse_theta<2, false>));
        g_static_ptr[dev] = ptr;
    }
    *out = g_static_ptr[dev];
    return AFQMC_OK;
}

size_t align256(size_t b) { return (b + 255) & ~(size_t)255; }

}  // namespace

extern "C" int afqmc_log_overlap_static(const void *trial, const void *walkers, int N, int n_alpha, int n_beta, int n_walkers,
                                        void *out_overlaps, void *stream_) {
    if (!trial || !walkers || !out_overlaps) return fail(nullptr, AFQMC_ERR_ARG, "afqmc_log_overlap_static: null pointer argument");
    if (N < 1 || n_walkers < 1 || n_alpha < 0 || n_beta < 0 || n_alpha > N || n_beta > N || n_alpha + n_beta < 1)
        return fail(nullptr, AFQMC_ERR_ARG, "afqmc_log_overlap_static: size out of range (N=%d n_alpha=%d n_beta=%d n_walkers=%d)", N, n_alpha,
                    n_beta, n_walkers);
    if (n_alpha > AFQMC_MAX_NOCC || n_beta > AFQMC_MAX_NOCC)
        return fail(nullptr, AFQMC_ERR_UNSUPPORTED, "afqmc_log_overlap_static: n_sigma > %d is not supported", AFQMC_MAX_NOCC);
    if (int rc = check_arch(nullptr, nullptr)) return rc;
    cudaStream_t stream = (cudaStream_t)stream_;
    const int ns[2] = {n_alpha, n_beta};
    const int nmax = std::max(n_alpha, n_beta), ksteps = (N + 3) / 4, kpad = 8 * ((N + K1_ROWS - 1) / K1_ROWS);

    // ---- carve the scratch: [zero block n_max x N][per spin: Re plane, Im plane][per spin: theta][e1][logdet] -------------------
    size_t off = 0, plane_bytes[2], theta_bytes[2], plane_off[2][2], theta_off[2];
    const size_t zero_off = off;
    off += align256((size_t)nmax * N * 8);
    for (int s = 0; s < 2; ++s) {
        plane_bytes[s] = (size_t)kpad * ((ns[s] + 7) / 8) * 32 * 8;
        for (int pl = 0; pl < 2; ++pl) { plane_off[s][pl] = off; off += align256(plane_bytes[s]); }
    }
    const size_t clear_bytes = off;                                   // everything up to here must start at zero
    for (int s = 0; s < 2; ++s) {
        theta_bytes[s] = (size_t)n_walkers * ((2 * ns[s] + 7) / 8) * ksteps * 32 * 8;
        theta_off[s] = off; off += align256(theta_bytes[s]);
    }
    const size_t e1_off = off; off += align256((size_t)2 * n_walkers * 16);
    const size_t ld_off = off; off += align256((size_t)2 * n_walkers * 16);
    if (off > (size_t)AFQMC_STATIC_SCRATCH_BYTES)
        return fail(nullptr, AFQMC_ERR_UNSUPPORTED,
                    "afqmc_log_overlap_static: N=%d n_alpha=%d n_beta=%d n_walkers=%d needs %zu bytes of scratch, the static array holds %d "
                    "(use afqmc_create / afqmc_local_energy for larger batches)", N, n_alpha, n_beta, n_walkers, off, AFQMC_STATIC_SCRATCH_BYTES);
    unsigned char *base = nullptr;
    if (int rc = static_scratch_for_current_device(&base)) return rc;

    // ---- the array keeps the last call's contents: clear the zero block and the fragment planes (their padding) -----------------
    CU_TRY(nullptr, cudaMemsetAsync(base, 0, clear_bytes, stream));
    size_t toff = 0;
    for (int s = 0; s < 2; ++s) {
        if (ns[s] == 0) continue;
        k11_pack_trial<<<(N * ns[s] + 255) / 256, 256, 0, stream>>>(reinterpret_cast<const double2 *>(trial) + toff, N, ns[s],
                                                                   reinterpret_cast<double *>(base + plane_off[s][0]),
                                                                   reinterpret_cast<double *>(base + plane_off[s][1]));
        CU_TRY(nullptr, cudaGetLastError());
        toff += (size_t)N * ns[s];
    }

    // ---- K1 as it stands (k1_overlap.cuh), complex-trial path (an all-zero Im plane adds exact zeros), theta into the scratch ----
    K1Params p1{};
    p1.walkers = reinterpret_cast<const double2 *>(walkers);
    p1.n_walkers = n_walkers; p1.N = N; p1.maxw = n_walkers; p1.spin0 = 0; p1.w0 = 0;
    p1.spin_off[0] = 0; p1.spin_off[1] = (long long)n_walkers * N * n_alpha;
    size_t k1s = 0;
    for (int s = 0; s < 2; ++s) {
        p1.n[s] = ns[s];
        if (ns[s] == 0) continue;
        p1.psiA[s] = reinterpret_cast<const double *>(base + plane_off[s][0]);
        p1.psiA_im[s] = reinterpret_cast<const double *>(base + plane_off[s][1]);
        p1.ht[s] = p1.ht_im[s] = reinterpret_cast<const double *>(base + zero_off);
        p1.thetaB[s] = reinterpret_cast<double *>(base + theta_off[s]);
        const int strips = (2 * ns[s] + 7) / 8;
        p1.layB[s] = OperandLayout{ns[s], strips, ksteps, 1, (long long)strips * ksteps * 32};      // one walker per tile
        k1s = std::max(k1s, (size_t)k1_layout(ns[s], true).total);
    }
    p1.e1 = reinterpret_cast<double *>(base + e1_off);
    p1.logdet = reinterpret_cast<double *>(base + ld_off);
    const int size = nmax <= 32 ? 0 : (2 * (k1s + 1024) <= 233472 ? 1 : 2);
    const dim3 grid(n_walkers, 2);
    if (size == 2) k1_overlap_inverse_theta<2, false><<<grid, K1_THREADS, k1s, stream>>>(p1);
    else if (size == 1) k1_overlap_inverse_theta<1, false><<<grid, K1_THREADS, k1s, stream>>>(p1);
    else k1_overlap_inverse_theta<0, false><<<grid, K1_THREADS, k1s, stream>>>(p1);
    CU_TRY(nullptr, cudaGetLastError());
    k8_log_overlap<<<(n_walkers + 127) / 128, 128, 0, stream>>>(n_walkers, n_walkers, n_alpha, n_beta, p1.logdet, reinterpret_cast<double *>(out_overlaps));
    CU_TRY(nullptr, cudaGetLastError());
    return AFQMC_OK;
}
