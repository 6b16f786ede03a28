// phoebe_elph.cu -- C ABI (include/phoebe_elph.h) and host-side orchestration of the
// sm_100a kernels for the el-ph Wannier->Bloch |g|^2 hot path (Eq. 7, 13, 70, 71).
// No CPU fallback: every compute call fails with PHOEBE_ELPH_E_CUDA without a device.
#include "../../include/phoebe_elph.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <array>
#include <map>
#include <mutex>
#include <string>
#include <vector>

#include "contract_planar.cuh"
#include "contract_pair.cuh"
#include "qfold.cuh"
#include "contract_i8.cuh"
#include "qbatch_kernels.cuh"
#include "rotate_v3.cuh"
#include "setk_kernels.cuh"
#include "setk_pair.cuh"

namespace {

constexpr int kSMs = 148;                 // B200
constexpr size_t kAlign = 256;
constexpr int kQPad = 128;                // q columns of Pt are padded to this (largest BM)
constexpr int kKPad = 16;                 // phase matrices are zero padded to this many rows (largest KC)
constexpr int kKBatchMax = 32;            // most k-points per set_k_batch (largest BM of the a1 GEMM)
constexpr int kMaxG = 4096;                // most reciprocal lattice vectors of the polar G sum (f4)
constexpr size_t kCBytesCap = 9000000000ull;   // C + Pt of one q sub-batch (whole batch whenever it fits)

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
int ceil_div(int a, int b) { return (a + b - 1) / b; }

// ---- set_k launch geometry --------------------------------------------------
int setk_threads(int X)
{
    for (int t = 256; t >= 64; t -= 32)
        if (X % t == 0) return t;
    if (X < 256) return (int)align_up((size_t)X, 32);
    return 256;
}
int setk_auto_split(int nRe, int nRp, int X)
{
    const int T = setk_threads(X);
    const long base = (long)nRp * ceil_div(X, T);
    long S = (kSMs * 12 + base - 1) / base;
    const long cap = std::max(1, nRe / 16);
    S = std::max(1L, std::min(S, std::min(16L, cap)));
    return (int)S;
}

// ---- workspace layout ---------------------------------------------------------
struct Layout {
    int Kpad = 0, KpadE = 0, ldq = 0, nq_sub = 0, S_alloc = 0, nk_slots = 1;
    size_t g1_stride = 0;   // complex elements between the g1' of consecutive k slots
    size_t g1P_stride = 0;  // doubles between the planar blocked copies of g1' (k_contract_planar) of consecutive k slots
    // contract_i8.cuh: bytes of one digit plane of A (all q tiles) and of B' (one k slot), rows padded to 64, columns to 64
    int i8_Kpad = 0, i8_Npad2 = 0, i8_ldsb = 0;
    size_t i8_a_plane = 0, i8_b_plane = 0;
    size_t off_Re = 0, off_Rp = 0, off_dege = 0, off_degp = 0, off_Uk = 0, off_kdev = 0, off_Ptk = 0, off_pairE = 0, off_zero = 0, off_Tpart = 0,
           off_g1 = 0, off_g1P = 0, off_pair = 0, off_Pt = 0, off_PtP = 0, off_C = 0, off_part = 0, off_fold = 0, off_Ai8 = 0, off_Bi8 = 0, off_sb = 0, off_rate = 0, off_seps = 0, off_G = 0, off_Zstar = 0, off_P = 0, off_sq = 0, off_sUkq = 0, off_sev = 0, off_som = 0, off_sout = 0, total = 0;
    size_t sz_sq = 0, sz_sUkq = 0, sz_sev = 0, sz_som = 0, sz_sout = 0;   // bytes of ONE staging slot (there are two)
};

// complex elements of C per q-point in the layout rotate_v3.cuh reads (row pitch P >= nm, b1 block pitch PB <= nw*P + 7)
size_t c_elems_per_q(const phoebe_elph_dims& d, int nb1)
{
    return (size_t)nb1 * ((size_t)d.nw * pe::rot3_row_pitch(d.nmodes) + 7);
}

int default_nq_sub(const phoebe_elph_dims& d, int nq_max)
{
    const size_t per_q = 16 * (c_elems_per_q(d, d.nb1_max) + (size_t)d.nRp + 4);
    long n = (long)(kCBytesCap / per_q);
    n = n / kQPad * kQPad;
    n = std::max<long>(n, kQPad);
    n = std::min<long>(n, (long)align_up((size_t)nq_max, kQPad));
    return (int)n;
}

Layout make_layout(const phoebe_elph_dims& d, int nq_max)
{
    Layout L;
    const size_t X = (size_t)d.nw * d.nw * d.nmodes;
    const size_t N = (size_t)d.nb1_max * d.nw * d.nmodes;
    L.Kpad = (int)align_up((size_t)d.nRp, kKPad);     // k_contract: Kpad % KC == 0 for every KC in use
    L.KpadE = (int)align_up((size_t)d.nRe, kKPad);
    L.nk_slots = std::max(1, d.nk_max);
    L.g1_stride = align_up((size_t)d.nRp * N, 16);
    L.nq_sub = default_nq_sub(d, nq_max);
    L.ldq = L.nq_sub;
    const int S_auto = setk_auto_split(d.nRe, d.nRp, (int)X);
    const int cap = std::max(1, std::min(16, d.nRe / 16));
    L.S_alloc = ((size_t)cap * d.nRp * X * 16 <= (256ull << 20)) ? std::max(cap, S_auto) : S_auto;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, kAlign); return o; };
    L.off_Re = take((size_t)d.nRe * 3 * 8);
    L.off_Rp = take((size_t)d.nRp * 3 * 8);
    L.off_dege = take((size_t)d.nRe * 8);
    L.off_degp = take((size_t)d.nRp * 8);
    L.off_Uk = take((size_t)L.nk_slots * d.nw * d.nb1_max * 16);
    L.off_kdev = take((size_t)kKBatchMax * 3 * 8);
    L.off_Ptk = take((size_t)(L.KpadE + 16) * kKBatchMax * 16);
    // +R / -R pair map of the Re list for the a1 GEMM (setk_pair.cuh): row map (2 ints) + vector + weight per pair
    L.off_pairE = take((size_t)(d.nRe + 8) * (2 * 4 + 4 * 8));
    L.off_zero = take(X * 16);                                       // a row of zeros (vectors without partner)
    L.off_Tpart = take((size_t)std::max(L.S_alloc, L.nk_slots) * d.nRp * X * 16);
    L.off_g1 = take((size_t)L.nk_slots * L.g1_stride * 16);
    // planar blocked copies ([rows][tiles of 64][3][64] doubles) of g1' and of the phases for k_contract_planar
    L.g1P_stride = ((size_t)d.nRp * 192 + 1920) * ceil_div((int)N, 64);    // (+ 15 padding rows of the pair form)
    L.off_g1P = take((size_t)L.nk_slots * L.g1P_stride * 8);
    // +R / -R pair map of the Rp list for k_contract_pair: 3 int + 4 double per real row, at most 2 nRp rows
    L.off_pair = take((size_t)(2 * d.nRp + 16) * (3 * 4 + 4 * 8));
    L.off_Pt = take((size_t)L.Kpad * L.ldq * 16);
    L.off_PtP = take((size_t)L.Kpad * L.ldq * 24);
    L.off_C = take((size_t)L.nq_sub * c_elems_per_q(d, d.nb1_max) * 16);
    // f2: linewidth partials [nq][groups of b2 tiles][nb1], staging of rate / eps_k / eps_kq for the host entry point
    L.off_part = take((size_t)nq_max * ceil_div(d.nb2_max, 8) * d.nb1_max * 8);
    // a4 on the INT8 tensor cores (contract_i8.cuh): six digit planes of the phases and of the pair rows, column scales
    L.i8_Kpad = (int)align_up((size_t)(2 * d.nRp + 16), 64);                   // >= any Kr
    L.i8_Npad2 = (int)align_up(2 * N, 64);
    L.i8_ldsb = (int)align_up(N, 32);
    L.i8_a_plane = (size_t)L.ldq * L.i8_Kpad;
    L.i8_b_plane = (size_t)L.i8_Npad2 * L.i8_Kpad;
    L.off_Ai8 = take(6 * L.i8_a_plane);
    L.off_Bi8 = take((size_t)L.nk_slots * 6 * L.i8_b_plane);
    L.off_sb = take((size_t)2 * L.nk_slots * L.i8_ldsb * 8);      // column scales, then the column maxima they come from
    // q <-> -q fold: hash table (power of two >= 2 nq, so < 4 nq ints), partner / representative / mate lists, meta
    L.off_fold = take((size_t)nq_max * (7 * 4 + 8) + 512);
    L.off_rate = take((size_t)2 * 2 * L.nk_slots * d.nb1_max * 8);    // two slots of (rate, eps_k), each [k slots][nb1]
    L.off_seps = take((size_t)2 * nq_max * d.nb2_max * 8);            // two slots of eps_kq
    // f4: G list and Born charges of the polar term, its (q, nu) amplitudes
    L.off_G = take((size_t)kMaxG * 3 * 8);
    L.off_Zstar = take((size_t)ceil_div(d.nmodes, 3) * 9 * 8);
    L.off_P = take((size_t)nq_max * d.nmodes * 16);
    // staging for the host-buffer entry points
    // (two slots each: q_batch_host_async copies batch n+1 in and batch n-1 out while batch n computes)
    L.sz_sq = align_up((size_t)nq_max * 3 * 8, kAlign);
    L.sz_sUkq = align_up((size_t)nq_max * d.nw * d.nb2_max * 16, kAlign);
    L.sz_sev = align_up((size_t)nq_max * d.nmodes * d.nmodes * 16, kAlign);
    L.sz_som = align_up((size_t)nq_max * d.nmodes * 8, kAlign);
    L.sz_sout = align_up((size_t)nq_max * d.nb1_max * d.nb2_max * d.nmodes * 8, kAlign);
    L.off_sq = take(2 * L.sz_sq);
    L.off_sUkq = take(2 * L.sz_sUkq);
    L.off_sev = take(2 * L.sz_sev);
    L.off_som = take(2 * L.sz_som);
    L.off_sout = take(2 * L.sz_sout);
    L.total = off;
    return L;
}

bool dims_ok(const phoebe_elph_dims* d, bool need_nq)
{
    if (d->nRe <= 0 || d->nRp <= 0 || d->nw <= 0 || d->nmodes <= 0) return false;
    if (d->nb1_max <= 0 || d->nb1_max > d->nw || d->nb2_max <= 0 || d->nb2_max > d->nw) return false;
    if (d->nq_max < 0 || (need_nq && d->nq_max == 0)) return false;
    if (d->nk_max < 0 || d->nk_max > kKBatchMax) return false;
    if (d->nRp > 32768 || d->nRe > 65535) return false;     // grid.y / grid.z limits of the kernels (pair rows <= 1.5 nRp)
    if (d->nmodes > 48 && d->nq_max > 0 && (size_t)d->nq_max > ((size_t)1 << 30)) return false;
    if ((long)d->nw * d->nw * d->nmodes > (1L << 24)) return false;
    return true;
}

struct EventPair { int kind; cudaEvent_t a, b; };

}  // namespace

struct phoebe_elph_ctx {
    phoebe_elph_dims dims{};
    const double2* gW = nullptr;
    cudaStream_t stream = nullptr;
    char* ws = nullptr;
    size_t ws_bytes = 0;
    Layout L;
    double *Re = nullptr, *Rp = nullptr, *deg_e = nullptr, *deg_p = nullptr;
    double *kdev = nullptr;
    double2 *Uk = nullptr, *Ptk = nullptr, *Tpart = nullptr, *g1_base = nullptr, *g1 = nullptr, *Pt = nullptr, *C = nullptr;
    int nb1 = 0;
    int nk_have = 0;        // k slots filled by the last set_k / set_k_batch
    bool have_k = false;
    int nq_sub = 0, s_split = 0;
    bool m3 = true;           // tuning "m3": three-multiply complex product (3 DMMA per tile and k-step instead of 4)
    int tile = 0;             // tuning "tile": 0 = automatic, 32 / 64 = force the contraction tile
    bool rot_plain = false;   // tuning "rot_plain": force the DFMA rotation kernel
    int rot_blk = 0;          // tuning "rot_blk": U_kq / ev staging of the rotation kernel: 0 automatic, 1 row copies, 2 one block per q
    int rot_qg = 0, rot_gb1 = 0, rot_mtw = 0;   // tuning "rot_qg" / "rot_gb1" / "rot_mtw": override the v2 rotation geometry (0 = automatic)
    int64_t launches[PHOEBE_ELPH_K_COUNT] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    bool qfold = false;       // tuning "qfold" (opt-in): contract (q, -q) pairs of a q list once (qfold.cuh)
    int i8 = 1;               // tuning "i8": 1 = a4 on the INT8 tensor cores by exact digit splitting (contract_i8.cuh), 0 = FP64 DMMA
    bool Bi8_stale = true;    // the digit planes of g1' must be rebuilt (as g1P_stale)
    double i8_scaleA = 2.0;   // power-of-two scale of the phase matrix: 2 x the largest weight 1/deg_p, rounded up
    int last_i8 = -1;
    int i8_cluster = 0;       // tuning "i8_cluster": 0 = choose, 1 / 2 / 4 / 8 = CTAs per cluster of the INT8 contraction (A planes multicast)
    int last_i8_cluster = 0, last_i8_grid = 0;
    bool last_fold = false;   // the last contraction went through the fold-capable launch sequence
    // q_batch_host_async: copy-in / copy-out streams and the events that chain them to the compute stream
    cudaStream_t s_in = nullptr, s_out = nullptr;
    cudaEvent_t ev_in[2] = {nullptr, nullptr}, ev_done[2] = {nullptr, nullptr}, ev_out[2] = {nullptr, nullptr};
    bool async_ready = false;
    unsigned async_n = 0;
    // f4: polar long-range term (Eq. 14-15); nG == 0 = off
    int nG = 0;
    pe::PolarParams polar{};
    // set_conventions: sign of both Fourier phases and which of the three rotation matrices enter conjugated
    double phase_sign = 1.0;
    bool conj_Uk = false, conj_Ukq = true, conj_ev = false;
    double *g1P = nullptr, *PtP = nullptr;   // planar blocked operands of k_contract_planar
    bool planar = true;       // tuning "planar": a4 through k_contract_planar (default) or k_contract
    // k_contract_pair: the Rp list folded into Kr real rows (pair_Kr == 0: not usable); g1P then holds the pair form
    int pair_Kr = 0, pair_KrPad = 0, pair_K2 = 0;   // K2 = (cos, sin) row pairs
    int pair_Kc = 0, pair_Kc4 = 0;                  // cosine rows (pairs + self-inverse vectors), padded to a multiple of 4
    bool rp_integer = false;
    // a1 pair form (setk_pair.cuh): the Re list folded into npairE (cos, sin) row pairs; 0 = not usable
    int npairE = 0;
    int* pairE_rowmap = nullptr; double *pairE_R = nullptr, *pairE_w = nullptr; double2* zero_row = nullptr;
    bool setk_pair = true;    // tuning "setk_pair": 1 = use it when it saves tensor work (default), 0 = never
    bool last_setk_pair = false;
    int pair = 1;             // tuning "pair": 1 = use it when 4 Kr < 6 nRp (default), 0 = never, 2 = whenever the map exists
    int pair_ctas = 1;        // tuning "pair_ctas": persistent CTAs of k_contract_pair per SM (its ring is 100 KB: two fit)
    int last_pair = -1;       // did the last contraction launch use the pair form (-1: no launch yet)
    int g1P_form = 0;         // what g1P holds: 0 nothing, 1 planar (re, im, re+im), 2 pair rows (re, im)
    int *pair_pa = nullptr, *pair_pb = nullptr, *pair_kind = nullptr;
    double *pair_R = nullptr, *pair_w = nullptr;
    bool g1P_stale = true;    // canonical g1' changed (set_k, or handed out by g1_buffer) since the last pack
    int k_sel = 0;            // k slot chosen by select_k (its U_k is needed for the overlap of Eq. 15)
    bool prof = false;
    std::vector<EventPair> evs;
    std::vector<cudaEvent_t> ev_pool;
    std::string err;
};

namespace {

int fail(phoebe_elph_ctx* c, int code, const char* msg)
{
    if (c) c->err = msg;
    return code;
}
int cuda_fail(phoebe_elph_ctx* c, cudaError_t e, const char* what)
{
    if (c) { c->err = std::string(what) + ": " + cudaGetErrorString(e); }
    return PHOEBE_ELPH_E_CUDA;
}
#define PE_CUDA(ctx, expr)                                              \
    do {                                                                \
        cudaError_t _e = (expr);                                        \
        if (_e != cudaSuccess) return cuda_fail((ctx), _e, #expr);      \
    } while (0)

cudaEvent_t get_event(phoebe_elph_ctx* c)
{
    if (!c->ev_pool.empty()) { cudaEvent_t e = c->ev_pool.back(); c->ev_pool.pop_back(); return e; }
    cudaEvent_t e = nullptr;
    if (cudaEventCreate(&e) != cudaSuccess) return nullptr;
    return e;
}
struct LaunchScope {          // counts the launch and, when profiling, brackets it with events
    phoebe_elph_ctx* c; int kind; cudaEvent_t b = nullptr;
    LaunchScope(phoebe_elph_ctx* c_, int kind_) : c(c_), kind(kind_)
    {
        c->launches[kind]++;
        if (c->prof) {
            cudaEvent_t a = get_event(c); b = get_event(c);
            if (a && b) {
                cudaEventRecord(a, c->stream);
                c->evs.push_back({kind, a, b});
            } else {                       // out of events: this launch goes untimed
                if (a) c->ev_pool.push_back(a);
                if (b) c->ev_pool.push_back(b);
                b = nullptr;
            }
        }
    }
    ~LaunchScope() { if (b) cudaEventRecord(b, c->stream); }
};

// Per-device function attributes (the shared-memory opt-in is per device, not per context): set once per
// (device, kernel, size), behind a mutex -- contexts on several threads share the table.
cudaError_t ensure_smem_optin(const void* kern, size_t bytes)
{
    static std::mutex mu;
    static std::map<std::pair<int, const void*>, size_t> done;
    if (bytes <= (48u << 10)) return cudaSuccess;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lock(mu);
    size_t& have = done[{dev, kern}];
    if (have >= bytes) return cudaSuccess;
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess) have = bytes;
    return e;
}

// ---- batched complex GEMM launcher (a4 and multi-k a1) ------------------------------
struct GemmArgs {
    const double2* At; int lda; const double2* B; int ldb; long long strideB;
    double2* C; long long ldc; long long strideC; int M, N, K, Kpad, batch;
    int rowsPerB = 0, rowOffset = 0; long long strideBrow = 0;      // multi-k a4: B slab switches every rowsPerB rows
    pe::CMap cm{0, 0, 0, 0};                                        // a4: column -> offset map of the C layout (ptx_helpers.cuh)
};
template <int BM, int BN, int WM, int WN, int KC, int ST, bool M3, int MINB = 1>
cudaError_t launch_contract(cudaStream_t stream, const GemmArgs& g, bool persistent = true)
{
    using Cfg = pe::ContractCfg<BM, BN, WM, WN, KC, ST>;
    auto kern = pe::k_contract<BM, BN, WM, WN, KC, ST, M3, MINB>;
    // per instantiation AND per device (the shared-memory opt-in is a per-device function attribute); contexts on
    // several threads share the table
    static std::mutex mu;
    static int ctas_by_dev[64] = {0};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) dev = 0;
    int ctas_per_sm;
    {
        std::lock_guard<std::mutex> lock(mu);
        if (ctas_by_dev[dev] == 0) {
            cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::kSmemBytes);
            if (e != cudaSuccess) return e;
            int nb = 0;
            e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kern, Cfg::kThreads, Cfg::kSmemBytes);
            if (e != cudaSuccess) return e;
            ctas_by_dev[dev] = std::max(1, nb);
        }
        ctas_per_sm = ctas_by_dev[dev];
    }
    // persistent grid: one CTA per resident slot, each walks the tile list with stride gridDim.x
    const long long ntiles = (long long)ceil_div(g.N, BN) * ceil_div(g.M, BM) * g.batch;
    // (the HBM-streaming multi-k a1 GEMM measured faster with one tile per CTA: the next CTA's prologue keeps
    //  loads in flight while this one stores; it passes persistent = false)
    if (ntiles > 0x7fffffffLL) return cudaErrorInvalidValue;
    const int grid = persistent ? (int)std::min<long long>(ntiles, (long long)kSMs * ctas_per_sm) : (int)ntiles;
    // persistent grid: panels as wide as the grid (each CTA keeps one column tile per panel, B panel L2-resident);
    // one-tile-per-CTA grid: plain n-fastest order
    const int panelW = persistent ? grid : 0x7fffffff;
    kern<<<grid, Cfg::kThreads, Cfg::kSmemBytes, stream>>>(g.At, g.lda, g.B, g.ldb, g.strideB, g.C, g.ldc, g.strideC,
                                                           g.M, g.N, g.K, g.Kpad, g.batch, g.rowsPerB, g.rowOffset,
                                                           g.strideBrow, panelW, g.cm);
    return cudaGetLastError();
}

int launch_setk_rotate(phoebe_elph_ctx* c, const double2* T, int S, const double2* Uk_dev, int nb1, double2* g1,
                       int nk, long long strideT, long long strideG)
{
    const phoebe_elph_dims& d = c->dims;
    const int Y = d.nw * d.nmodes, N = nb1 * Y;
    LaunchScope ls(c, PHOEBE_ELPH_K_SETK_ROTATE);
    // threads per block over y: the largest of 128 / 64 / 32 that leaves the fewest idle threads in the last block
    // (Y = 192 -> 64: three full blocks instead of one and a half; Y = 48 -> 64 instead of 128)
    int TR = 128;
    for (int t : {64, 32})
        if (ceil_div(Y, t) * t < ceil_div(Y, TR) * TR) TR = t;
    if (nb1 <= 4) {
        const int ng = ceil_div(nb1, 4);
        dim3 grid(ceil_div(Y, TR), d.nRp, ng * nk);
        pe::k_setk_rotate<4><<<grid, TR, (size_t)d.nw * 4 * 16, c->stream>>>(T, Uk_dev, S, d.nRp, d.nw, Y, nb1, g1, N, ng,
                                                                             strideT, strideG, c->conj_Uk ? 1 : 0);
    } else if (nb1 <= 8) {
        const int ng = ceil_div(nb1, 8);
        dim3 grid(ceil_div(Y, TR), d.nRp, ng * nk);
        pe::k_setk_rotate<8><<<grid, TR, (size_t)d.nw * 8 * 16, c->stream>>>(T, Uk_dev, S, d.nRp, d.nw, Y, nb1, g1, N, ng,
                                                                             strideT, strideG, c->conj_Uk ? 1 : 0);
    } else {
        const int ng = ceil_div(nb1, 16);
        dim3 grid(ceil_div(Y, TR), d.nRp, ng * nk);
        pe::k_setk_rotate<16><<<grid, TR, (size_t)d.nw * 16 * 16, c->stream>>>(T, Uk_dev, S, d.nRp, d.nw, Y, nb1, g1, N,
                                                                               ng, strideT, strideG, c->conj_Uk ? 1 : 0);
    }
    PE_CUDA(c, cudaGetLastError());
    return PHOEBE_ELPH_OK;
}

// U_k of every k slot is kept in the context (the overlap [U_kq^dagger U_k] of the polar term needs it at q_batch time)
int keep_Uk(phoebe_elph_ctx* c, const double2* Uk_dev, int nk, int nb1)
{
    if (Uk_dev != c->Uk)
        PE_CUDA(c, cudaMemcpyAsync(c->Uk, Uk_dev, (size_t)nk * c->dims.nw * nb1 * 16, cudaMemcpyDeviceToDevice, c->stream));
    return PHOEBE_ELPH_OK;
}

int run_set_k(phoebe_elph_ctx* c, const double* k, const double2* Uk_dev, int nb1)
{
    const phoebe_elph_dims& d = c->dims;
    if (int rc = keep_Uk(c, Uk_dev, 1, nb1)) return rc;
    const int X = d.nw * d.nw * d.nmodes;
    const int T = setk_threads(X);
    int S = c->s_split > 0 ? c->s_split : setk_auto_split(d.nRe, d.nRp, X);
    S = std::min(S, c->L.S_alloc);
    const int epc = ceil_div(d.nRe, S);
    S = ceil_div(d.nRe, epc);
    if ((size_t)epc * 16 > (size_t)(227u << 10)) return fail(c, PHOEBE_ELPH_E_DIMS, "set_k: nRe too large for one Re chunk (raise s_split)");
    PE_CUDA(c, ensure_smem_optin((const void*)pe::k_setk_stream, (size_t)epc * 16));
    {
        LaunchScope ls(c, PHOEBE_ELPH_K_SETK_STREAM);
        dim3 grid(ceil_div(X, T), S, d.nRp);
        pe::k_setk_stream<<<grid, T, (size_t)epc * 16, c->stream>>>(c->gW, c->Re, c->deg_e, c->phase_sign * k[0], c->phase_sign * k[1], c->phase_sign * k[2], d.nRe,
                                                                    d.nRp, X, epc, c->Tpart);
        PE_CUDA(c, cudaGetLastError());
    }
    int rc = launch_setk_rotate(c, c->Tpart, S, Uk_dev, nb1, c->g1_base, 1, 0, 0);
    if (rc) return rc;
    c->nb1 = nb1;
    c->nk_have = 1;
    c->g1P_stale = true;
    c->Bi8_stale = true;
    c->k_sel = 0;
    c->g1 = c->g1_base;
    c->have_k = true;
    return PHOEBE_ELPH_OK;
}

// a1 for a batch of k-points in ONE pass over g_W: per phonon vector p a
// [nk x nRe].[nRe x X] complex GEMM on the FP64 tensor cores, then a2 per k.
int run_set_k_batch(phoebe_elph_ctx* c, int nk, const double* k_host, const double2* Uk_dev, int nb1)
{
    const phoebe_elph_dims& d = c->dims;
    const int X = d.nw * d.nw * d.nmodes;
    if (int rc = keep_Uk(c, Uk_dev, nk, nb1)) return rc;
    PE_CUDA(c, cudaMemcpyAsync(c->kdev, k_host, (size_t)nk * 24, cudaMemcpyHostToDevice, c->stream));
    // the fold pays where the three-multiply GEMM is FP64-bound (6 nk flop per 16 bytes of g_W against 37 TFLOP/s and
    // 6.5 TB/s: nk >= 12; measured: 32 k band-window 0.306 -> 0.201 ms, 16 k 4-atom 4.93 -> 4.69 ms, 4 k large cell
    // 8.1 -> 9.4 ms -- HBM-bound, where the plain form streams better)
    c->last_setk_pair = c->setk_pair && c->m3 && c->npairE > 0 && nk >= 12;
    if (c->last_setk_pair) {
        // +R / -R pairs of the Re list folded (setk_pair.cuh): real phases x complex sums formed on the fly
        const int Kr = 2 * c->npairE, KrPad = (int)align_up((size_t)Kr, 8);
        double* PtkR = reinterpret_cast<double*>(c->Ptk);
        {
            LaunchScope ls(c, PHOEBE_ELPH_K_QPHASE);
            pe::k_kphase_pair<<<dim3(1, std::min(KrPad / 2, 256)), 32, 0, c->stream>>>(c->kdev, c->pairE_R, c->pairE_w, nk, c->npairE,
                                                                                      KrPad, c->phase_sign, PtkR);
            PE_CUDA(c, cudaGetLastError());
        }
        {
            LaunchScope ls(c, PHOEBE_ELPH_K_SETK_GEMM);
            const int grid = ceil_div(X, 128) * d.nRp;
            auto launch = [&](auto kern, size_t smem, int threads) -> cudaError_t {
                cudaError_t e2 = ensure_smem_optin((const void*)kern, smem);
                if (e2 != cudaSuccess) return e2;
                kern<<<grid, threads, smem, c->stream>>>(PtkR, c->gW, (long long)d.nRe * X, X, c->pairE_rowmap, c->zero_row, c->Tpart,
                                                         (long long)d.nRp * X, nk, Kr, KrPad, d.nRp);
                return cudaGetLastError();
            };
            cudaError_t e;
            // ring depth 4 (72 KB per CTA: three CTAs per SM); measured on the 4-atom cell (16 k): 4 / 6 / 8 stages of 8 rows ->
            // 3.92 / 4.70 / 7.50 ms, 3 / 4 stages of 16 rows -> 4.42 / 6.44 ms: resident CTAs matter more than ring depth
#ifndef PHOEBE_SETKP_ST
#define PHOEBE_SETKP_ST 4
#endif
            constexpr int ST = PHOEBE_SETKP_ST;
            if (nk <= 8) e = launch(pe::k_setk_pair<8, 128, 4, 8, ST>, pe::SetkPairCfg<8, 128, 4, 8, ST>::kSmemBytes, 160);
            else if (nk <= 16) e = launch(pe::k_setk_pair<16, 128, 4, 8, ST>, pe::SetkPairCfg<16, 128, 4, 8, ST>::kSmemBytes, 160);
            else e = launch(pe::k_setk_pair<32, 128, 4, 8, ST + 1>, pe::SetkPairCfg<32, 128, 4, 8, ST + 1>::kSmemBytes, 160);   // band-window, 32 k: 3 / 4 / 5 stages -> 0.223 / 0.205 / 0.201 ms
            PE_CUDA(c, e);
        }
    } else {
    {
        LaunchScope ls(c, PHOEBE_ELPH_K_QPHASE);
        dim3 grid(1, std::min(c->L.KpadE, 256));
        pe::k_qphase<<<grid, 32, 0, c->stream>>>(c->kdev, c->Re, c->deg_e, nk, d.nRe, c->L.KpadE, kKBatchMax, c->Ptk,
                                                 c->phase_sign, nullptr);
        PE_CUDA(c, cudaGetLastError());
    }
    {
        LaunchScope ls(c, PHOEBE_ELPH_K_SETK_GEMM);
        GemmArgs g{c->Ptk, kKBatchMax, c->gW, X, (long long)d.nRe * X, c->Tpart, (long long)d.nRp * X, (long long)X,
                   nk, X, d.nRe, c->L.KpadE, d.nRp};
        cudaError_t e;
        if (c->m3) {
            if (nk <= 8) e = launch_contract<8, 128, 1, 4, 8, 4, true>(c->stream, g, false);
            // 6 ring stages: the deepest ring that still leaves two CTAs per SM (2 x 114 KB); measured on the 4-atom cell
            // 4 / 5 / 6 / 8 stages -> 5.06 / 5.03 / 4.93 / 6.79 ms
            else if (nk <= 16) e = launch_contract<16, 128, 1, 4, 8, 6, true>(c->stream, g, false);
            else e = launch_contract<32, 128, 1, 8, 8, 4, true>(c->stream, g, false);
        } else {
            if (nk <= 8) e = launch_contract<8, 128, 1, 4, 8, 4, false>(c->stream, g, false);
            else if (nk <= 16) e = launch_contract<16, 128, 1, 4, 8, 4, false>(c->stream, g, false);
            else e = launch_contract<32, 128, 1, 4, 8, 4, false>(c->stream, g, false);
        }
        PE_CUDA(c, e);
    }
    }
    {
        int rc = launch_setk_rotate(c, c->Tpart, 1, Uk_dev, nb1, c->g1_base, nk, (long long)d.nRp * X,
                                    (long long)c->L.g1_stride);
        if (rc) return rc;
    }
    c->nb1 = nb1;
    c->nk_have = nk;
    c->g1P_stale = true;
    c->Bi8_stale = true;
    c->k_sel = 0;
    c->g1 = c->g1_base;
    c->have_k = true;
    return PHOEBE_ELPH_OK;
}

// ---- k_rotate_v3<KS, GB, MTW, RATES> (rotate_v3.cuh): KS = ceil(nm/4) in 1..12, GB = b1 per warp item, MTW = tiles of b2 ----
// GB per KS: the smallest that fills whole a5 column tiles (2 for odd KS <= 3, else 1) or, when nb1 allows, the largest
// whose accumulators fit (a U_kq / ev fragment then feeds GB x as many tensor instructions).
int rot3_min_gb(int KS) { return (KS == 1 || KS == 3) ? 2 : 1; }
int rot3_max_gb(int KS, int MTW)
{
    if (MTW == 1) return KS == 1 ? 8 : KS == 2 ? 4 : (KS == 3 || KS == 4) ? 2 : 1;
    return KS == 1 ? 4 : (KS == 2 || KS == 3) ? 2 : 1;
}
// the instantiations live in rot3_instances.cu (four translation units by KS range)
extern "C" const void* pe_rot3_kernel_part0(int KS, int GB, int MTW, int mode);
extern "C" const void* pe_rot3_kernel_part1(int KS, int GB, int MTW, int mode);
extern "C" const void* pe_rot3_kernel_part2(int KS, int GB, int MTW, int mode);
extern "C" const void* pe_rot3_kernel_part3(int KS, int GB, int MTW, int mode);
const void* rot3_kernel(int KS, int GB, int MTW, int mode)     // mode: 0 plain, 1 linewidths (f2), 3 polar (f4)
{
    if (KS <= 2) return pe_rot3_kernel_part0(KS, GB, MTW, mode);
    if (KS <= 5) return pe_rot3_kernel_part1(KS, GB, MTW, mode);
    if (KS <= 9) return pe_rot3_kernel_part2(KS, GB, MTW, mode);
    return pe_rot3_kernel_part3(KS, GB, MTW, mode);
}

// geometry of one rotation launch
struct Rot3Geom { int KS, GB, MTW, P, PB, QS, gb1, nmg, blk; size_t smem; };
constexpr size_t kRot3SmemBudget = 200u << 10;

bool rot3_geometry(int nw, int nm, int nb1, int nb2, int nq, bool rates, int qs_over, int gb1_over, int mtw_over,
                   int blk_over, Rot3Geom* G)
{
    const int KS = ceil_div(nm, 4), NT = ceil_div(nm, 8), MT = ceil_div(nb2, 8);
    G->KS = KS;
    // two tiles of b2 per item (8 consumer warps with ~230 registers) when an item has many a5 column tiles to share
    // each A fragment over (KS >= 5: the large cell 7.28 vs 7.78 ms per launch); else one tile and 12 consumer warps
    // (the 4-atom cell: 3.27 vs 3.57 ms)
    G->MTW = (mtw_over > 0) ? ((mtw_over >= 2 && MT >= 2) ? 2 : 1) : ((MT >= 2 && KS >= 5) ? 2 : 1);
    G->GB = nb1 >= rot3_max_gb(KS, G->MTW) ? rot3_max_gb(KS, G->MTW) : rot3_min_gb(KS);
    G->nmg = ceil_div(MT, G->MTW);
    G->P = pe::rot3_row_pitch(nm);
    // a5 column tiles that hold pairs of two different b1 (GB >= 2, odd KS): b1 block pitch = 4 mod 8 keeps their B
    // fragment loads conflict-free
    const int raw = nw * G->P;
    G->PB = raw + ((G->GB >= 2 && (KS & 1)) ? ((4 - raw % 8) + 8) % 8 : 0);
    // U_kq / ev as one block per q-point when their nw + nm row copies (~80 clocks of the TMA unit each) would weigh
    // more than half of the q-point's tensor work (4 clocks per DMMA): the small cells
    const long dmma_q = 3L * ceil_div(nb1, G->GB) * G->nmg * G->MTW *
                        ((long)ceil_div(G->GB * KS, 2) * ceil_div(nw, 4) + (long)G->GB * KS * NT);
    G->blk = blk_over > 0 ? blk_over - 1 : (long)(nw + nm) * 80 > 2 * dmma_q;
    auto total = [&](int QS, int gb1) { return (size_t)pe::rot3_layout(nw, nm, nb2, G->PB, QS, gb1, rates, G->blk != 0).total; };
    if (G->blk && nb1 * G->PB > 8192) G->blk = 0;                  // (block mode is for whole-q stages)
    int qs_cap = std::max(1, 128 / (8 * std::max(NT, MT)));            // the producer lanes' register slots
    if (G->blk) qs_cap = std::min(qs_cap, 32);                         // one lane per q-point's block copy
    if (total(1, nb1) <= kRot3SmemBudget && gb1_over <= 0) {
        // whole q-points per stage: enough of them that every consumer warp has an item, while the q list still
        // gives every SM several stages
        const int per_q = ceil_div(nb1, G->GB) * G->nmg;
        int QS = ceil_div(pe::rot3_consumers(G->MTW), per_q);
        if (qs_over > 0) QS = qs_over;
        QS = std::min(QS, qs_cap);
        while (QS > 1 && (total(QS, nb1) > kRot3SmemBudget || ceil_div(nq, QS) < 2 * kSMs)) --QS;
        G->QS = QS; G->gb1 = nb1;
    } else {
        int gb1 = 0;
        for (int cand = nb1; cand >= 1; --cand) {
            if (cand % G->GB) continue;
            if (total(1, cand) <= kRot3SmemBudget) { gb1 = cand; break; }
        }
        if (gb1 == 0) {
            if (total(1, 1) > (size_t)(227u << 10) - 1024) return false;
            gb1 = 1;
        }
        // no larger than gives every consumer warp one item (smaller stages: deeper prefetch for the same memory)
        const int want = std::max(G->GB, ceil_div(pe::rot3_consumers(G->MTW), G->nmg) * G->GB);
        gb1 = std::min(gb1, std::max(want, G->GB));
        if (gb1_over > 0) gb1 = std::min(gb1_over, nb1);
        G->QS = 1; G->gb1 = std::min(gb1, nb1);
    }
    G->smem = total(G->QS, G->gb1);
    return G->smem <= (size_t)(227u << 10);
}

struct RateReq {           // f2: linewidth accumulation fused into the epilogue (nullptr = plain q_batch)
    const double* eps_k; const double* eps_kq; phoebe_elph_rate_params prm; double* rate;
};

// rows_per_k > 0: the q lists of the k slots slot0, slot0+1, .. are stacked (nq = slots * rows_per_k rows); row block j uses
// the g1' of slot slot0 + j
int run_q_batch(phoebe_elph_ctx* c, int nq, int nb2, const double* q, const double2* Ukq, const double2* ev,
                const double* omega, double* out, const RateReq* rr = nullptr, int rows_per_k = 0, int slot0 = 0)
{
    const phoebe_elph_dims& d = c->dims;
    const int nb1 = c->nb1, Y = d.nw * d.nmodes, N = nb1 * Y;
    const int nq_sub = std::min(c->nq_sub, c->L.nq_sub);
    // rotation kernel geometry: rotate_v3 (FP64 tensor cores) for nm <= 48, else the plain DFMA kernel
    const bool polar = c->nG > 0;
    Rot3Geom G{};
    // (a cell whose U_kq / ev stages do not fit three-deep in shared memory -- nw beyond ~56 -- takes the plain kernel too)
    const bool use_mma = d.nmodes <= 48 && !c->rot_plain &&
                         rot3_geometry(d.nw, d.nmodes, nb1, nb2, std::min(nq, nq_sub), rr != nullptr || polar, c->rot_qg, c->rot_gb1,
                                       c->rot_mtw, c->rot_blk, &G);
    const bool fused_rates = rr != nullptr && use_mma;
    int gb1 = nb1, rot_threads = 0;
    size_t rot_smem = 0;
    int P = d.nmodes, PB = d.nw * d.nmodes;                 // C layout (plain for the DFMA kernel)
    if (use_mma) {
        // (the polar kernels, mode 3, always carry the Eq. 29 arrays in their stages)
        P = G.P; PB = G.PB; gb1 = G.gb1; rot_smem = G.smem; rot_threads = pe::rot3_threads(G.MTW);
    } else {
        const size_t fixed = ((size_t)d.nw * nb2 + (size_t)d.nmodes * d.nmodes) * 16;
        const size_t per_b1 = ((size_t)Y + (size_t)nb2 * d.nmodes) * 16;
        gb1 = (int)std::max<size_t>(1, std::min<size_t>((size_t)nb1, ((96u << 10) - std::min<size_t>(fixed, 90u << 10)) / per_b1));
        rot_smem = fixed + per_b1 * gb1;
        if (rot_smem > (200u << 10)) return fail(c, PHOEBE_ELPH_E_DIMS, "rotation tile does not fit shared memory");
        const int work = gb1 * nb2 * d.nmodes;
        rot_threads = std::max(32, std::min(256, (int)align_up((size_t)work, 32)));
    }
    const long long ldcq = (long long)nb1 * PB;            // complex elements of C per q-point
    const pe::CMap cm = (P == d.nmodes && PB == d.nw * d.nmodes) ? pe::CMap{0, 0, 0, 0}
                                                                   : pe::CMap{d.nmodes, d.nw, P, PB - d.nw * P};
    double2* Pbuf = reinterpret_cast<double2*>(c->ws + c->L.off_P);
    pe::PolarArgs pa{nullptr, c->Uk + (size_t)c->k_sel * d.nw * nb1, (c->conj_Ukq ? 0 : 1) | (c->conj_ev ? 2 : 0)};
    double* plain_scratch = nullptr;
    if (rr && !use_mma && out == nullptr) {     // the plain path sums from the stored |g|^2: its own scratch behind C
        if ((size_t)std::min(nq, nq_sub) * (size_t)ldcq * 16 + (size_t)std::min(nq, nq_sub) * nb1 * nb2 * d.nmodes * 8 >
            (size_t)c->L.nq_sub * c_elems_per_q(d, d.nb1_max) * 16)
            return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_rates without out: not available for nmodes > 48 at this size");
        plain_scratch = reinterpret_cast<double*>(c->C + (size_t)std::min(nq, nq_sub) * ldcq);
    }
    const void* rot_kernel = use_mma ? rot3_kernel(G.KS, G.GB, G.MTW, polar ? 3 : fused_rates ? 1 : 0)
                                     : (const void*)pe::k_rotate_epilogue;
    if (!rot_kernel) return fail(c, PHOEBE_ELPH_E_DIMS, "no rotation kernel for this mode count");
    double* partial = reinterpret_cast<double*>(c->ws + c->L.off_part);
    pe::RateArgs ra{nullptr, nullptr, 0.0, 0.0, 0.0, partial, 0};
    if (rr && rows_per_k > 0) {
        if (!use_mma) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_rates_multi: not available for nmodes > 48");
        if (nq > nq_sub) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_rates_multi: the stacked batch must fit one contraction launch (fewer k slots)");
        ra.rows_per_k = rows_per_k;
    }
    if (rr) {
        ra.eps_k = rr->eps_k;
        ra.inv_kT = 1.0 / rr->prm.kT;
        ra.mu = rr->prm.mu;
        ra.inv_sigma2 = 1.0 / (rr->prm.sigma * rr->prm.sigma);
    }
    PE_CUDA(c, ensure_smem_optin(rot_kernel, rot_smem));

    for (int qs = 0; qs < nq; qs += nq_sub) {
        const int nqs = std::min(nq_sub, nq - qs);
        const int ncols = (int)align_up((size_t)nqs, kQPad);
        // contraction tile: 64x64 unless that leaves the 148 SMs with a long ragged tail (few tiles);
        // cost model = rounds of tiles per SM x tile area (+5 % for the smaller tile's extra operand traffic)
        // (the 64 x 64 tile is the one with the +R / -R pair form: 4 instead of 6 real flop per MAC)
        const bool pair_ok = c->m3 && c->planar && c->pair_Kr > 0 &&
                             (c->pair == 2 || (c->pair == 1 && (size_t)4 * c->pair_Kr < (size_t)6 * d.nRp));
        const double cost64 = (double)ceil_div(ceil_div(nqs, 64) * ceil_div(N, 64), kSMs) * 64 * 64 *
                              (pair_ok ? 4.0 * c->pair_Kr / (6.0 * d.nRp) : 1.0);
        const double cost32 = (double)ceil_div(ceil_div(nqs, 32) * ceil_div(N, 32), kSMs) * 32 * 32 * 1.05;
        int tile = c->tile > 0 ? c->tile : (cost32 < cost64 ? 32 : 64);
        if (rows_per_k > 0 && tile != 32 && tile != 64) tile = 64;       // the stacked form knows these two tiles
        const bool use_planar = c->m3 && c->planar && tile == 64;
        // +R / -R pairs folded (contract_pair.cuh): real phases x complex pair rows, 4 real flop per MAC instead of 6
        const bool use_pair = use_planar && c->pair_Kr > 0 &&
                              (c->pair == 2 || (c->pair == 1 && (size_t)4 * c->pair_Kr < (size_t)6 * d.nRp));
        c->last_pair = use_pair ? 1 : 0;
        // the pair form on the INT8 tensor cores by exact digit splitting (contract_i8.cuh)
        const bool use_i8 = use_pair && c->i8 != 0 && !(c->qfold && rows_per_k == 0 && nqs >= 256) &&
                            (rows_per_k == 0 || rows_per_k % pe::I8Cfg::BM == 0) &&    // a row tile must not straddle two k slots
                            c->pair_Kr <= 16384;      // exact INT32 accumulation: 6 digit pairs x rows x 128^2 < 2^31
        c->last_i8 = use_i8 ? 1 : 0;
        const int i8_Kpad = (int)align_up((size_t)c->pair_Kr, pe::I8Cfg::KC), i8_Npad2 = (int)align_up((size_t)2 * N, 64);
        int8_t* Ai8 = reinterpret_cast<int8_t*>(c->ws + c->L.off_Ai8);
        int8_t* Bi8 = reinterpret_cast<int8_t*>(c->ws + c->L.off_Bi8);
        double* sbv = reinterpret_cast<double*>(c->ws + c->L.off_sb);
        if (use_i8 && c->Bi8_stale) {
            LaunchScope ls(c, PHOEBE_ELPH_K_PACK);
            unsigned long long* cmax = reinterpret_cast<unsigned long long*>(sbv + (size_t)c->L.nk_slots * c->L.i8_ldsb);
            PE_CUDA(c, cudaMemsetAsync(cmax, 0, (size_t)c->nk_have * c->L.i8_ldsb * 8, c->stream));
            pe::k_i8_colmax<<<dim3(ceil_div(N, 128), ceil_div(c->pair_Kr, 16), c->nk_have), 128, 0, c->stream>>>(
                c->g1_base, (long long)N, (long long)c->L.g1_stride, N, c->pair_Kr, c->pair_pa, c->pair_pb, c->pair_kind, cmax, c->L.i8_ldsb);
            PE_CUDA(c, cudaGetLastError());
            pe::k_pack_i8<<<dim3(ceil_div(i8_Npad2, 128), i8_Kpad / 16, c->nk_have), 128, 0, c->stream>>>(
                c->g1_base, (long long)N, (long long)c->L.g1_stride, N, i8_Npad2, c->pair_Kr, i8_Kpad, c->pair_pa, c->pair_pb,
                c->pair_kind, cmax, sbv, c->L.i8_ldsb, Bi8, 6 * c->L.i8_b_plane);
            PE_CUDA(c, cudaGetLastError());
            c->Bi8_stale = false;
        }
        if (use_planar && !use_i8 && (c->g1P_stale || c->g1P_form != (use_pair ? 2 : 1))) {
            // canonical g1' of every filled k slot -> blocked operand copy (planar planes, or pair rows)
            LaunchScope ls(c, PHOEBE_ELPH_K_PACK);
            if (use_pair) {
                dim3 grid(ceil_div(N, 64), c->pair_Kr, c->nk_have);
                pe::k_pack_pair<<<grid, 64, 0, c->stream>>>(c->g1_base, (long long)N, (long long)c->L.g1_stride, N, c->pair_pa,
                                                            c->pair_pb, c->pair_kind, c->g1P, (long long)c->L.g1P_stride);
            } else {
                dim3 grid(ceil_div(N, 64), d.nRp, c->nk_have);
                pe::k_pack_planar<<<grid, 64, 0, c->stream>>>(c->g1_base, (long long)N, (long long)c->L.g1_stride, N, c->g1P,
                                                              (long long)c->L.g1P_stride);
            }
            PE_CUDA(c, cudaGetLastError());
            c->g1P_stale = false;
            c->g1P_form = use_pair ? 2 : 1;
        }
        // q <-> -q fold (qfold.cuh): the pairs are found on the device; both launch sequences are enqueued and the
        // kernels of the path not taken return at once
        const bool try_fold = use_pair && !use_i8 && c->qfold && rows_per_k == 0 && nqs >= 256 && c->pair_K2 > 0;
        int* fold_base = reinterpret_cast<int*>(c->ws + c->L.off_fold);
        int tsize = 1;
        while (tsize < 2 * nqs) tsize <<= 1;
        int* f_meta = fold_base;                 // [2] (+ padding)
        int* f_partner = fold_base + 64;
        int* f_rep = f_partner + nqs;
        int* f_mate = f_rep + nqs;
        int* f_table = f_mate + nqs;             // [tsize] < 4 nqs
        unsigned long long* f_fp = reinterpret_cast<unsigned long long*>(
            c->ws + c->L.off_fold + align_up((size_t)(64 + 3 * (size_t)nqs + tsize) * 4, 8));
        pe::FoldArgs fa{nullptr, nullptr, nullptr, 0};
        c->last_fold = try_fold;
        if (try_fold) {
            LaunchScope ls(c, PHOEBE_ELPH_K_QFOLD);
            const bool in_smem = nqs <= 8192;                  // fingerprints + table + partners: nq (8 + 4) + 4 tsize bytes
            const size_t dsm = in_smem ? (size_t)nqs * 12 + (size_t)tsize * 4 : 0;
            PE_CUDA(c, ensure_smem_optin((const void*)pe::k_qfold_detect, dsm));
            pe::k_qfold_detect<<<1, 1024, dsm, c->stream>>>(q + 3 * (size_t)qs, nqs, c->rp_integer ? 1 : 0, in_smem ? 1 : 0, f_table,
                                                            tsize, f_partner, f_fp, f_rep, f_mate, f_meta);
            PE_CUDA(c, cudaGetLastError());
            fa = pe::FoldArgs{f_meta, f_rep, f_mate, c->pair_Kc4};
        }
        {
            LaunchScope ls(c, PHOEBE_ELPH_K_QPHASE);
            if (use_i8) {
                pe::k_qphase_i8<<<dim3(ceil_div(ncols, 128), c->pair_Kc4 / 16), 128, 0, c->stream>>>(
                    q + 3 * (size_t)qs, c->pair_R, c->pair_w, c->pair_K2, c->pair_Kc, c->pair_Kc4, nqs, i8_Kpad, c->L.ldq,
                    c->phase_sign, 1.0 / c->i8_scaleA, Ai8);
            } else if (use_pair) {
                dim3 grid(ceil_div(ncols, 256), std::min(c->pair_Kc4, 64));
                pe::k_qphase_pair<<<grid, 256, 0, c->stream>>>(q + 3 * (size_t)qs, c->pair_R, c->pair_w, c->pair_K2, c->pair_Kc,
                                                               c->pair_Kc4, nqs, c->pair_Kr, c->pair_KrPad, c->L.ldq,
                                                               c->phase_sign, c->PtP, nullptr, nullptr, fa.meta ? fa.meta + 1 : nullptr, 0);
                if (try_fold) {      // the same over the representatives only
                    PE_CUDA(c, cudaGetLastError());
                    pe::k_qphase_pair<<<grid, 256, 0, c->stream>>>(q + 3 * (size_t)qs, c->pair_R, c->pair_w, c->pair_K2, c->pair_Kc,
                                                                   c->pair_Kc4, nqs, c->pair_Kr, c->pair_KrPad, c->L.ldq,
                                                                   c->phase_sign, c->PtP, f_rep, f_meta, f_meta + 1, 1);
                }
            } else {
                dim3 grid(ceil_div(ncols, 256), std::min(c->L.Kpad, 64));
                pe::k_qphase<<<grid, 256, 0, c->stream>>>(q + 3 * (size_t)qs, c->Rp, c->deg_p, nqs, d.nRp, c->L.Kpad,
                                                          c->L.ldq, c->Pt, c->phase_sign, use_planar ? c->PtP : nullptr);
            }
            PE_CUDA(c, cudaGetLastError());
        }
        {
            LaunchScope ls(c, PHOEBE_ELPH_K_CONTRACT);
            GemmArgs g{c->Pt, c->L.ldq, c->g1, N, 0, c->C, ldcq, 0, nqs, N, d.nRp, c->L.Kpad, 1};
            g.cm = cm;
            if (rows_per_k > 0) {
                g.B = c->g1_base + (size_t)slot0 * c->L.g1_stride; g.rowsPerB = rows_per_k; g.rowOffset = qs;
                g.strideBrow = (long long)c->L.g1_stride;
            }
            if (use_i8) {
                // clusters of CL CTAs share the A digit planes of a row tile by multicast (contract_i8.cuh): tuning "i8_cluster"
                const int ntm8 = ceil_div(nqs, pe::I8Cfg::BM), ntn8 = ceil_div(2 * N, pe::I8Cfg::BN);
                int CL = c->i8_cluster;
                if (CL != 1 && CL != 2 && CL != 4 && CL != 8) CL = 1;       // measured (4-atom, band-window, large): 2 and 4 change nothing; 8 is 12 % faster per CTA but only 15 clusters (120 CTAs) fit
                const void* kfn = CL == 8 ? (const void*)pe::k_contract_i8<8> : CL == 4 ? (const void*)pe::k_contract_i8<4>
                                : CL == 2 ? (const void*)pe::k_contract_i8<2> : (const void*)pe::k_contract_i8<1>;
                PE_CUDA(c, ensure_smem_optin(kfn, pe::I8Cfg::kSmemBytes));
                const int ngroups = ntm8 * ceil_div(ntn8, CL);
                cudaLaunchConfig_t cfg = {};
                cfg.blockDim = dim3(pe::I8Cfg::kThreads);
                cfg.dynamicSmemBytes = pe::I8Cfg::kSmemBytes;
                cfg.stream = c->stream;
                cudaLaunchAttribute attr[1];
                attr[0].id = cudaLaunchAttributeClusterDimension;
                attr[0].val.clusterDim.x = CL; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
                cfg.attrs = attr; cfg.numAttrs = CL > 1 ? 1 : 0;
                int nclusters = kSMs / CL;
                if (CL > 1) {           // clusters that can be resident at once (a GPC's SM count need not be a multiple of CL)
                    cfg.gridDim = dim3(kSMs / CL * CL);
                    int nc = 0;
                    PE_CUDA(c, cudaOccupancyMaxActiveClusters(&nc, kfn, &cfg));
                    if (nc > 0) nclusters = std::min(nclusters, nc);
                }
                cfg.gridDim = dim3(std::min(ngroups, nclusters) * CL);
                const int8_t* Bi8s = Bi8 + (size_t)(rows_per_k > 0 ? slot0 : c->k_sel) * 6 * c->L.i8_b_plane;
                const double* sbs = sbv + (size_t)(rows_per_k > 0 ? slot0 : c->k_sel) * c->L.i8_ldsb;
                const int8_t* Ai8c = Ai8;
                size_t b_sl = 6 * c->L.i8_b_plane;
                int ldsb = c->L.i8_ldsb, Mi = nqs, Ni = N, Kp = i8_Kpad, rpk = rows_per_k, ro = qs;
                double sA = c->i8_scaleA;
                double2* Cp = c->C;
                long long ldc8 = ldcq;
                pe::CMap cm8 = cm;
                void* kargs[] = {&Ai8c, &Bi8s, &b_sl, &sbs, &ldsb, &sA, &Cp, &ldc8, &Mi, &Ni, &Kp, &rpk, &ro, &cm8};
                PE_CUDA(c, cudaLaunchKernelExC(&cfg, kfn, kargs));
                c->last_i8_cluster = CL;
                c->last_i8_grid = (int)cfg.gridDim.x;
            } else if (use_pair) {
                PE_CUDA(c, ensure_smem_optin((const void*)pe::k_contract_pair<false>, pe::PairCfg::kSmemBytes));
                const int ntiles = ceil_div(nqs, 64) * ceil_div(N, 64);
                const int grid = std::min(ntiles, kSMs * c->pair_ctas);
                const int slot = rows_per_k > 0 ? slot0 : c->k_sel;
                int panelW = grid;      // as for the planar form: the panel of pair rows (width x Kr x 1024 B) stays in L2
                while (panelW % 2 == 0 && (size_t)panelW * c->pair_Kr * pe::PairCfg::ROWB * 8 > (48u << 20)) panelW /= 2;
                pe::k_contract_pair<false><<<grid, pe::PairCfg::kThreads, pe::PairCfg::kSmemBytes, c->stream>>>(
                    c->PtP, c->L.ldq, c->g1P + (size_t)slot * c->L.g1P_stride, ceil_div(N, 64), (long long)c->L.g1P_stride,
                    c->C, ldcq, nqs, N, c->pair_Kr, c->pair_KrPad, rows_per_k, qs, panelW, cm, fa);
                PE_CUDA(c, cudaGetLastError());
                if (try_fold) {
                    PE_CUDA(c, ensure_smem_optin((const void*)pe::k_contract_pair<true>, pe::PairCfg::kFoldSmemBytes));
                    pe::k_contract_pair<true><<<grid, pe::PairCfg::kThreads, pe::PairCfg::kFoldSmemBytes, c->stream>>>(
                        c->PtP, c->L.ldq, c->g1P + (size_t)slot * c->L.g1P_stride, ceil_div(N, 64), (long long)c->L.g1P_stride,
                        c->C, ldcq, nqs, N, c->pair_Kr, c->pair_KrPad, 0, 0, panelW, cm, fa);
                    PE_CUDA(c, cudaGetLastError());
                }
            } else if (use_planar) {
                PE_CUDA(c, ensure_smem_optin((const void*)pe::k_contract_planar, pe::PlanarCfg::kSmemBytes));
                const int ntiles = ceil_div(nqs, 64) * ceil_div(N, 64);
                const int grid = std::min(ntiles, kSMs);
                const int slot = rows_per_k > 0 ? slot0 : c->k_sel;
                // panel width: a divisor of the grid (each CTA keeps its column tile for a whole panel) small enough
                // that the panel of g1P (width x K x 1536 B) stays L2-resident next to the streaming phase rows and C
                int panelW = grid;
                while (panelW % 2 == 0 && (size_t)panelW * d.nRp * pe::PlanarCfg::ROW * 8 > (48u << 20)) panelW /= 2;
                pe::k_contract_planar<<<grid, pe::PlanarCfg::kThreads, pe::PlanarCfg::kSmemBytes, c->stream>>>(
                    c->PtP, c->L.ldq / 64, c->g1P + (size_t)slot * c->L.g1P_stride, ceil_div(N, 64),
                    (long long)c->L.g1P_stride, c->C, ldcq, nqs, N, d.nRp, c->L.Kpad, rows_per_k, qs, panelW, cm);
                PE_CUDA(c, cudaGetLastError());
            } else if (c->m3) {
                if (tile == 32) PE_CUDA(c, (launch_contract<32, 32, 2, 2, 16, 3, true>(c->stream, g)));
                else PE_CUDA(c, (launch_contract<64, 64, 2, 4, 16, 4, true>(c->stream, g)));
            } else {
                if (tile == 32) PE_CUDA(c, (launch_contract<32, 32, 2, 2, 16, 3, false>(c->stream, g)));
                else PE_CUDA(c, (launch_contract<64, 64, 2, 2, 16, 3, false, 2>(c->stream, g)));
            }
        }
        if (polar) {
            LaunchScope ls(c, PHOEBE_ELPH_K_POLAR);
            pe::k_polar_amp<<<ceil_div(nqs, 4), 128, (size_t)4 * d.nmodes * 8, c->stream>>>(
                q + 3 * (size_t)qs, ev + (size_t)qs * d.nmodes * d.nmodes, reinterpret_cast<const double*>(c->ws + c->L.off_G),
                reinterpret_cast<const double*>(c->ws + c->L.off_Zstar), nqs, d.nmodes, c->nG, c->polar, Pbuf);
            PE_CUDA(c, cudaGetLastError());
            pa.P = Pbuf;
        }
        if (rr) ra.eps_kq = rr->eps_kq + (size_t)qs * nb2;
        double* op = out ? out + (size_t)qs * nb1 * nb2 * d.nmodes : nullptr;
        {
            LaunchScope ls(c, PHOEBE_ELPH_K_ROTATE_EPI);
            const double2* Up = Ukq + (size_t)qs * d.nw * nb2;
            const double2* Zp = ev + (size_t)qs * d.nmodes * d.nmodes;
            const double* wp = omega + (size_t)qs * d.nmodes;
            if (use_mma) {
                // persistent: one CTA per SM walks the groups of QS q-points
                pe::Rot3Args ar{c->C, Up, Zp, wp, op, nqs, d.nw, d.nmodes, nb1, nb2, PB, G.QS, G.gb1, G.blk, ra, pa};
                if (rows_per_k > 0) ar.ra.eps_k = ra.eps_k + (size_t)(qs / rows_per_k) * nb1;   // (qs is 0 in the stacked rates form)
                void* args[] = {&ar};
                const int grid = std::min(ceil_div(nqs, G.QS), kSMs);
                PE_CUDA(c, cudaLaunchKernel(rot_kernel, dim3(grid), dim3(rot_threads), args, rot_smem, c->stream));
            } else {
                if (plain_scratch) op = plain_scratch;
                const double2* Cp = c->C; long long ldc = ldcq;
                int nw_ = d.nw, nm_ = d.nmodes, nb1_ = nb1, nb2_ = nb2, gb1_ = gb1, P_ = P, PB_ = PB;
                void* args[] = {&Cp, &ldc, &P_, &PB_, &Up, &Zp, &wp, &op, &nw_, &nm_, &nb1_, &nb2_, &gb1_, &pa};
                for (int y0 = 0; y0 < nqs; y0 += 65535) {          // grid.y limit
                    const int ny = std::min(65535, nqs - y0);
                    const double2* Cy = c->C + (size_t)y0 * ldcq; const double2* Uy = Up + (size_t)y0 * d.nw * nb2;
                    const double2* Zy = Zp + (size_t)y0 * d.nmodes * d.nmodes; const double* wy = wp + (size_t)y0 * d.nmodes;
                    double* oy = op + (size_t)y0 * nb1 * nb2 * d.nmodes;
                    pe::PolarArgs pay = pa;
                    if (pay.P) pay.P += (size_t)y0 * d.nmodes;
                    args[0] = &Cy; args[4] = &Uy; args[5] = &Zy; args[6] = &wy; args[7] = &oy; args[13] = &pay;
                    PE_CUDA(c, cudaLaunchKernel(rot_kernel, dim3(ceil_div(nb1, gb1), ny), dim3(rot_threads), args, rot_smem,
                                                c->stream));
                }
            }
        }
        if (rr) {
            int nparts = nqs * G.nmg;                   // rotate_v3: one partial row per (q, group of b2 tiles)
            if (!use_mma) {        // plain rotation path: sum from the stored |g|^2, 32 q per warp
                const int QC = 32;
                nparts = ceil_div(nqs, QC);
                LaunchScope ls(c, PHOEBE_ELPH_K_ROTATE_EPI);
                pe::k_rates_from_out<<<dim3(nparts, nb1), 32, 0, c->stream>>>(op, omega + (size_t)qs * d.nmodes, nqs, d.nmodes,
                                                                              nb1, nb2, QC, ra);
                PE_CUDA(c, cudaGetLastError());
            }
            LaunchScope ls(c, PHOEBE_ELPH_K_RATE_REDUCE);
            const double scale = rr->prm.pref / (sqrt(3.14159265358979323846) * rr->prm.sigma);
            if (rows_per_k > 0)        // one (partial rows, rate[nb1]) block per k slot
                pe::k_rate_reduce<<<dim3(nb1, nq / rows_per_k), 256, 0, c->stream>>>(partial, rows_per_k * G.nmg, nb1, scale, rr->rate);
            else
                pe::k_rate_reduce<<<nb1, 256, 0, c->stream>>>(partial, nparts, nb1, scale, rr->rate);
            PE_CUDA(c, cudaGetLastError());
        }
    }
    return PHOEBE_ELPH_OK;
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// The synchronous host entry points use staging slot 0 on the compute stream: first let the copy-out stream
// finish with any batch q_batch_host_async still has in flight.
int drain_async(phoebe_elph_ctx* c)
{
    if (c->async_ready && c->async_n > 0) {
        PE_CUDA(c, cudaStreamSynchronize(c->stream));
        PE_CUDA(c, cudaStreamSynchronize(c->s_out));
        c->async_n = 0;
    }
    return PHOEBE_ELPH_OK;
}

}  // namespace

// =============================================================================
extern "C" {

const char* phoebe_elph_version(void) { return "phoebe-elph-b200 0.1 (sm_100a)"; }

int phoebe_elph_workspace_bytes(const phoebe_elph_dims* dims, size_t budget, size_t* bytes_out, int32_t* nq_batch_out)
{
    if (!dims || !bytes_out || !nq_batch_out) return PHOEBE_ELPH_E_NULL;
    if (!dims_ok(dims, false)) return PHOEBE_ELPH_E_DIMS;
    int hi = dims->nq_max > 0 ? dims->nq_max : (1 << 24);
    if (make_layout(*dims, 1).total > budget) return PHOEBE_ELPH_E_WORKSPACE;
    int lo = 1;                                   // invariant: layout(lo) fits
    if (make_layout(*dims, hi).total <= budget) lo = hi;
    while (lo < hi) {
        int mid = lo + (hi - lo + 1) / 2;
        if (make_layout(*dims, mid).total <= budget) lo = mid; else hi = mid - 1;
    }
    *nq_batch_out = lo;
    *bytes_out = make_layout(*dims, lo).total;
    return PHOEBE_ELPH_OK;
}

int phoebe_elph_setup(phoebe_elph_ctx** ctx_out, const void* gW_dev, const double* Re_host, const double* Rp_host,
                      const double* deg_e_host, const double* deg_p_host, const phoebe_elph_dims* dims,
                      void* workspace_dev, size_t workspace_bytes, void* cuda_stream)
{
    if (!ctx_out) return PHOEBE_ELPH_E_NULL;
    *ctx_out = nullptr;
    if (!gW_dev || !Re_host || !Rp_host || !dims || !workspace_dev) return PHOEBE_ELPH_E_NULL;
    if (!dims_ok(dims, true)) return PHOEBE_ELPH_E_DIMS;
    if (!aligned16(gW_dev) || (reinterpret_cast<uintptr_t>(workspace_dev) & (kAlign - 1))) return PHOEBE_ELPH_E_ALIGN;
    for (int i = 0; i < 3 * dims->nRe; ++i) if (!std::isfinite(Re_host[i])) return PHOEBE_ELPH_E_DIMS;
    for (int i = 0; i < 3 * dims->nRp; ++i) if (!std::isfinite(Rp_host[i])) return PHOEBE_ELPH_E_DIMS;
    for (int i = 0; deg_e_host && i < dims->nRe; ++i) if (!(deg_e_host[i] > 0.0)) return PHOEBE_ELPH_E_DIMS;
    for (int i = 0; deg_p_host && i < dims->nRp; ++i) if (!(deg_p_host[i] > 0.0)) return PHOEBE_ELPH_E_DIMS;
    Layout L = make_layout(*dims, dims->nq_max);
    if (L.total > workspace_bytes) return PHOEBE_ELPH_E_WORKSPACE;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return PHOEBE_ELPH_E_CUDA;

    phoebe_elph_ctx* c = new (std::nothrow) phoebe_elph_ctx();
    if (!c) return PHOEBE_ELPH_E_CUDA;
    c->dims = *dims;
    c->gW = static_cast<const double2*>(gW_dev);
    c->stream = static_cast<cudaStream_t>(cuda_stream);
    c->ws = static_cast<char*>(workspace_dev);
    c->ws_bytes = workspace_bytes;
    c->L = L;
    c->nq_sub = L.nq_sub;
    c->Re = reinterpret_cast<double*>(c->ws + L.off_Re);
    c->Rp = reinterpret_cast<double*>(c->ws + L.off_Rp);
    c->deg_e = reinterpret_cast<double*>(c->ws + L.off_dege);
    c->deg_p = reinterpret_cast<double*>(c->ws + L.off_degp);
    c->Uk = reinterpret_cast<double2*>(c->ws + L.off_Uk);
    c->Tpart = reinterpret_cast<double2*>(c->ws + L.off_Tpart);
    c->g1_base = reinterpret_cast<double2*>(c->ws + L.off_g1);
    c->g1 = c->g1_base;
    c->kdev = reinterpret_cast<double*>(c->ws + L.off_kdev);
    c->Ptk = reinterpret_cast<double2*>(c->ws + L.off_Ptk);
    c->Pt = reinterpret_cast<double2*>(c->ws + L.off_Pt);
    c->g1P = reinterpret_cast<double*>(c->ws + L.off_g1P);
    c->PtP = reinterpret_cast<double*>(c->ws + L.off_PtP);
    c->C = reinterpret_cast<double2*>(c->ws + L.off_C);

    std::vector<double> ones((size_t)std::max(dims->nRe, dims->nRp), 1.0);
    cudaError_t e = cudaSuccess;
    auto up = [&](void* dst, const void* src, size_t bytes) {
        if (e == cudaSuccess) e = cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, c->stream);
    };
    up(c->Re, Re_host, (size_t)dims->nRe * 24);
    up(c->Rp, Rp_host, (size_t)dims->nRp * 24);
    up(c->deg_e, deg_e_host ? deg_e_host : ones.data(), (size_t)dims->nRe * 8);
    up(c->deg_p, deg_p_host ? deg_p_host : ones.data(), (size_t)dims->nRp * 8);
    // ---- +R / -R pair map of the Rp list (contract_pair.cuh): a cosine block (one row per pair or vector without
    // partner, then one per self-inverse vector R = 0, zero rows up to a multiple of 4) and a sine block (one row per
    // pair, same order) ----
    std::vector<int> h_pa, h_pb, h_kind;
    std::vector<double> h_R, h_w;
    {
        const int nRp = dims->nRp;
        auto key = [&](int p, double sg) {
            return std::array<double, 3>{sg * Rp_host[3 * p] + 0.0, sg * Rp_host[3 * p + 1] + 0.0, sg * Rp_host[3 * p + 2] + 0.0};
        };
        auto wt = [&](int p) { return deg_p_host ? deg_p_host[p] : 1.0; };
        std::map<std::array<double, 3>, int> first;
        for (int p = nRp - 1; p >= 0; --p) first[key(p, 1.0)] = p;
        std::vector<char> used((size_t)nRp, 0);
        std::vector<int> selfs;
        auto row = [&](int a, int b, int kind) {
            h_pa.push_back(a); h_pb.push_back(b); h_kind.push_back(kind);
            h_R.push_back(Rp_host[3 * a]); h_R.push_back(Rp_host[3 * a + 1]); h_R.push_back(Rp_host[3 * a + 2]);
            h_w.push_back(1.0 / wt(a));
        };
        std::vector<std::pair<int, int>> pairs;
        for (int p = 0; p < nRp; ++p) {
            if (used[p]) continue;
            used[p] = 1;
            if (key(p, 1.0) == key(p, -1.0)) { selfs.push_back(p); continue; }
            int partner = -1;
            auto it = first.find(key(p, -1.0));
            if (it != first.end() && !used[it->second] && wt(it->second) == wt(p)) { partner = it->second; used[partner] = 1; }
            pairs.push_back({p, partner});
        }
        for (auto& pr : pairs) row(pr.first, pr.second, 0);
        c->pair_K2 = (int)pairs.size();
        for (int p : selfs) row(p, -1, 0);
        c->pair_Kc = (int)h_pa.size();
        while (h_pa.size() % 16) row(0, -1, 2);                 // zero rows: the sine block starts at a 16-row group (contract_i8.cuh)
        c->pair_Kc4 = (int)h_pa.size();
        for (auto& pr : pairs) row(pr.first, pr.second, 1);
        c->pair_Kr = (int)h_pa.size();
        {
            double wmax = 0.0;
            for (int p = 0; p < nRp; ++p) wmax = std::max(wmax, 1.0 / wt(p));
            int ex = 0;
            std::frexp(wmax, &ex);                               // wmax = f 2^ex, f in [1/2, 1)
            c->i8_scaleA = std::ldexp(1.0, ex + 1);              // |phase| <= wmax < 2^ex = scale / 2
        }
        c->rp_integer = true;                                   // q -> q + G leaves the phases alone only for integer Rp
        for (int i = 0; i < 3 * nRp; ++i) if (Rp_host[i] != std::floor(Rp_host[i])) c->rp_integer = false;
        c->pair_KrPad = (int)align_up((size_t)c->pair_Kr, (size_t)std::max(kKPad, pe::PairCfg::KC));
        // the pair form reuses the planar buffers: rows must fit them (g1P: Kr*128 <= nRp*192 doubles per tile column,
        // PtP: KrPad*8 <= Kpad*24 bytes per q)
        if ((size_t)c->pair_Kr * 128 > (size_t)nRp * 192 + 1920 || (size_t)c->pair_KrPad * 8 > (size_t)L.Kpad * 24) c->pair_Kr = 0;
        if (c->pair_Kr > 0) {
            char* base = c->ws + L.off_pair;
            const size_t cap = (size_t)2 * nRp + 16;
            c->pair_pa = reinterpret_cast<int*>(base);
            c->pair_pb = c->pair_pa + cap;
            c->pair_kind = c->pair_pb + cap;
            c->pair_R = reinterpret_cast<double*>(base + align_up(3 * cap * 4, 8));
            c->pair_w = c->pair_R + 3 * cap;
            up(c->pair_pa, h_pa.data(), h_pa.size() * 4);
            up(c->pair_pb, h_pb.data(), h_pb.size() * 4);
            up(c->pair_kind, h_kind.data(), h_kind.size() * 4);
            up(c->pair_R, h_R.data(), h_R.size() * 8);
            up(c->pair_w, h_w.data(), h_w.size() * 8);
        }
    }
    // ---- +R / -R pair map of the Re list (setk_pair.cuh): every vector is in exactly one "pair" (e, ebar | none) ----
    std::vector<int> hE_map;
    std::vector<double> hE_R, hE_w;
    {
        const int nRe = dims->nRe;
        auto key = [&](int p, double sg) {
            return std::array<double, 3>{sg * Re_host[3 * p] + 0.0, sg * Re_host[3 * p + 1] + 0.0, sg * Re_host[3 * p + 2] + 0.0};
        };
        auto wt = [&](int p) { return deg_e_host ? deg_e_host[p] : 1.0; };
        std::map<std::array<double, 3>, int> first;
        for (int p = nRe - 1; p >= 0; --p) first[key(p, 1.0)] = p;
        std::vector<char> used((size_t)nRe, 0);
        for (int p = 0; p < nRe; ++p) {
            if (used[p]) continue;
            used[p] = 1;
            int partner = -1;
            if (!(key(p, 1.0) == key(p, -1.0))) {
                auto it = first.find(key(p, -1.0));
                if (it != first.end() && !used[it->second] && wt(it->second) == wt(p)) { partner = it->second; used[partner] = 1; }
            }
            hE_map.push_back(p); hE_map.push_back(partner);
            hE_R.push_back(Re_host[3 * p]); hE_R.push_back(Re_host[3 * p + 1]); hE_R.push_back(Re_host[3 * p + 2]);
            hE_w.push_back(1.0 / wt(p));
        }
        const int P = (int)hE_w.size();
        // 2 DMMA per ring row x 2 P rows against 3 per row x nRe rows of the three-multiply form
        c->npairE = ((size_t)4 * P < (size_t)3 * nRe && 2 * P <= nRe + 8) ? P : 0;
        char* base = c->ws + L.off_pairE;
        c->pairE_rowmap = reinterpret_cast<int*>(base);
        c->pairE_R = reinterpret_cast<double*>(base + align_up((size_t)(nRe + 8) * 2 * 4, 8));
        c->pairE_w = c->pairE_R + 3 * (size_t)(nRe + 8);
        c->zero_row = reinterpret_cast<double2*>(c->ws + L.off_zero);
        if (c->npairE > 0) {
            up(c->pairE_rowmap, hE_map.data(), hE_map.size() * 4);
            up(c->pairE_R, hE_R.data(), hE_R.size() * 8);
            up(c->pairE_w, hE_w.data(), hE_w.size() * 8);
        }
        if (e == cudaSuccess)
            e = cudaMemsetAsync(c->zero_row, 0, (size_t)dims->nw * dims->nw * dims->nmodes * 16, c->stream);
    }
    // the 16-row groups of the A digit planes behind the sine block are read, never written (contract_i8.cuh)
    if (e == cudaSuccess) e = cudaMemsetAsync(c->ws + L.off_Ai8, 0, 6 * L.i8_a_plane, c->stream);
    // the padding elements of the C layout (rotate_v3.cuh) are read, never written: they must hold finite values
    if (e == cudaSuccess)
        e = cudaMemsetAsync(c->C, 0, (size_t)L.nq_sub * c_elems_per_q(*dims, dims->nb1_max) * 16, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) { delete c; return PHOEBE_ELPH_E_CUDA; }
    *ctx_out = c;
    return PHOEBE_ELPH_OK;
}

int phoebe_elph_set_k(phoebe_elph_ctx* c, const double* k_host, const void* Uk_dev, int32_t nb1)
{
    if (!c) return PHOEBE_ELPH_E_NULL;
    if (!k_host || !Uk_dev) return fail(c, PHOEBE_ELPH_E_NULL, "set_k: null pointer");
    if (nb1 <= 0 || nb1 > c->dims.nb1_max) return fail(c, PHOEBE_ELPH_E_DIMS, "set_k: nb1 out of range");
    if (!aligned16(Uk_dev)) return fail(c, PHOEBE_ELPH_E_ALIGN, "set_k: Uk not 16-byte aligned");
    return run_set_k(c, k_host, static_cast<const double2*>(Uk_dev), nb1);
}

int phoebe_elph_set_k_host(phoebe_elph_ctx* c, const double* k_host, const void* Uk_host, int32_t nb1)
{
    if (!c) return PHOEBE_ELPH_E_NULL;
    if (!k_host || !Uk_host) return fail(c, PHOEBE_ELPH_E_NULL, "set_k_host: null pointer");
    if (nb1 <= 0 || nb1 > c->dims.nb1_max) return fail(c, PHOEBE_ELPH_E_DIMS, "set_k_host: nb1 out of range");
    PE_CUDA(c, cudaMemcpyAsync(c->Uk, Uk_host, (size_t)c->dims.nw * nb1 * 16, cudaMemcpyHostToDevice, c->stream));
    return run_set_k(c, k_host, c->Uk, nb1);
}

int phoebe_elph_set_k_batch(phoebe_elph_ctx* c, int32_t nk, const double* k_host, const void* Uk_dev, int32_t nb1)
{
    if (!c) return PHOEBE_ELPH_E_NULL;
    if (!k_host || !Uk_dev) return fail(c, PHOEBE_ELPH_E_NULL, "set_k_batch: null pointer");
    if (nk <= 0 || nk > c->L.nk_slots) return fail(c, PHOEBE_ELPH_E_DIMS, "set_k_batch: nk out of range (dims.nk_max)");
    if (nb1 <= 0 || nb1 > c->dims.nb1_max) return fail(c, PHOEBE_ELPH_E_DIMS, "set_k_batch: nb1 out of range");
    if (!aligned16(Uk_dev)) return fail(c, PHOEBE_ELPH_E_ALIGN, "set_k_batch: Uk not 16-byte aligned");
    return run_set_k_batch(c, nk, k_host, static_cast<const double2*>(Uk_dev), nb1);
}

int phoebe_elph_set_k_batch_host(phoebe_elph_ctx* c, int32_t nk, const double* k_host, const void* Uk_host, int32_t nb1)
{
    if (!c) return PHOEBE_ELPH_E_NULL;
    if (!k_host || !Uk_host) return fail(c, PHOEBE_ELPH_E_NULL, "set_k_batch_host: null pointer");
    if (nk <= 0 || nk > c->L.nk_slots) return fail(c, PHOEBE_ELPH_E_DIMS, "set_k_batch_host: nk out of range (dims.nk_max)");
    if (nb1 <= 0 || nb1 > c->dims.nb1_max) return fail(c, PHOEBE_ELPH_E_DIMS, "set_k_batch_host: nb1 out of range");
    PE_CUDA(c, cudaMemcpyAsync(c->Uk, Uk_host, (size_t)nk * c->dims.nw * nb1 * 16, cudaMemcpyHostToDevice, c->stream));
    return run_set_k_batch(c, nk, k_host, c->Uk, nb1);
}

int phoebe_elph_select_k(phoebe_elph_ctx* c, int32_t i)
{
    if (!c) return PHOEBE_ELPH_E_NULL;
    if (!c->have_k) return fail(c, PHOEBE_ELPH_E_NO_K, "select_k before set_k / set_k_batch");
    if (i < 0 || i >= c->nk_have) return fail(c, PHOEBE_ELPH_E_DIMS, "select_k: index out of range");
    c->g1 = c->g1_base + (size_t)i * c->L.g1_stride;
    c->k_sel = i;
    return PHOEBE_ELPH_OK;
}

int phoebe_elph_q_batch(phoebe_elph_ctx* c, int32_t nq, int32_t nb2, const double* q_dev, const void* Ukq_dev,
                        const void* ev_dev, const double* omega_dev, double* out_dev)
{
    if (!c) return PHOEBE_ELPH_E_NULL;
    if (!c->have_k) return fail(c, PHOEBE_ELPH_E_NO_K, "q_batch before set_k");
    if (nq == 0) return PHOEBE_ELPH_OK;          // an empty batch is a no-op (nothing is read or written)
    if (!q_dev || !Ukq_dev || !ev_dev || !omega_dev || !out_dev) return fail(c, PHOEBE_ELPH_E_NULL, "q_batch: null pointer");
    if (nq < 0 || nq > c->dims.nq_max) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch: nq out of range");
    if (nb2 <= 0 || nb2 > c->dims.nb2_max) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch: nb2 out of range");
    if (!aligned16(Ukq_dev) || !aligned16(ev_dev)) return fail(c, PHOEBE_ELPH_E_ALIGN, "q_batch: complex input not 16-byte aligned");
    if ((reinterpret_cast<uintptr_t>(q_dev) | reinterpret_cast<uintptr_t>(omega_dev) | reinterpret_cast<uintptr_t>(out_dev)) & 7u)
        return fail(c, PHOEBE_ELPH_E_ALIGN, "q_batch: double array not 8-byte aligned");
    return run_q_batch(c, nq, nb2, q_dev, static_cast<const double2*>(Ukq_dev), static_cast<const double2*>(ev_dev),
                       omega_dev, out_dev);
}

int phoebe_elph_q_batch_multi(phoebe_elph_ctx* c, int32_t nk, int32_t nq, int32_t nb2, const double* q_dev,
                              const void* Ukq_dev, const void* ev_dev, const double* omega_dev, double* out_dev)
{
    if (!c) return PHOEBE_ELPH_E_NULL;
    if (!c->have_k) return fail(c, PHOEBE_ELPH_E_NO_K, "q_batch_multi before set_k_batch");
    if (!q_dev || !Ukq_dev || !ev_dev || !omega_dev || !out_dev) return fail(c, PHOEBE_ELPH_E_NULL, "q_batch_multi: null pointer");
    if (nk <= 0 || nk > c->nk_have) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_multi: nk exceeds the k slots of the last set_k_batch");
    if (nq < 0 || (nq % 64) != 0) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_multi: nq must be a multiple of 64");
    if (nq == 0) return PHOEBE_ELPH_OK;          // empty q lists: no-op
    if ((long long)nk * nq > c->dims.nq_max) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_multi: nk*nq exceeds nq_max");
    if (nb2 <= 0 || nb2 > c->dims.nb2_max) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_multi: nb2 out of range");
    if (c->nG > 0) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_multi: not available while the polar term is on");
    if (!aligned16(Ukq_dev) || !aligned16(ev_dev)) return fail(c, PHOEBE_ELPH_E_ALIGN, "q_batch_multi: complex input not 16-byte aligned");
    return run_q_batch(c, nk * nq, nb2, q_dev, static_cast<const double2*>(Ukq_dev), static_cast<const double2*>(ev_dev),
                       omega_dev, out_dev, nullptr, nq);
}

int phoebe_elph_q_batch_host(phoebe_elph_ctx* c, int32_t nq, int32_t nb2, const double* q_host, const void* Ukq_host,
                             const void* ev_host, const double* omega_host, double* out_host)
{
    if (!c) return PHOEBE_ELPH_E_NULL;
    if (!c->have_k) return fail(c, PHOEBE_ELPH_E_NO_K, "q_batch before set_k");
    if (nq == 0) return PHOEBE_ELPH_OK;          // an empty batch is a no-op (nothing is read or written)
    if (!q_host || !Ukq_host || !ev_host || !omega_host || !out_host) return fail(c, PHOEBE_ELPH_E_NULL, "q_batch_host: null pointer");
    if (nq < 0 || nq > c->dims.nq_max) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_host: nq out of range");
    if (nb2 <= 0 || nb2 > c->dims.nb2_max) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_host: nb2 out of range");
    if (int rc0 = drain_async(c)) return rc0;
    const phoebe_elph_dims& d = c->dims;
    double* sq = reinterpret_cast<double*>(c->ws + c->L.off_sq);
    double2* sU = reinterpret_cast<double2*>(c->ws + c->L.off_sUkq);
    double2* sZ = reinterpret_cast<double2*>(c->ws + c->L.off_sev);
    double* sw = reinterpret_cast<double*>(c->ws + c->L.off_som);
    double* so = reinterpret_cast<double*>(c->ws + c->L.off_sout);
    PE_CUDA(c, cudaMemcpyAsync(sq, q_host, (size_t)nq * 24, cudaMemcpyHostToDevice, c->stream));
    PE_CUDA(c, cudaMemcpyAsync(sU, Ukq_host, (size_t)nq * d.nw * nb2 * 16, cudaMemcpyHostToDevice, c->stream));
    PE_CUDA(c, cudaMemcpyAsync(sZ, ev_host, (size_t)nq * d.nmodes * d.nmodes * 16, cudaMemcpyHostToDevice, c->stream));
    PE_CUDA(c, cudaMemcpyAsync(sw, omega_host, (size_t)nq * d.nmodes * 8, cudaMemcpyHostToDevice, c->stream));
    int rc = run_q_batch(c, nq, nb2, sq, sU, sZ, sw, so);
    if (rc) return rc;
    PE_CUDA(c, cudaMemcpyAsync(out_host, so, (size_t)nq * c->nb1 * nb2 * d.nmodes * 8, cudaMemcpyDeviceToHost, c->stream));
    PE_CUDA(c, cudaStreamSynchronize(c->stream));
    return PHOEBE_ELPH_OK;
}

}  // extern "C"

namespace {
struct RateHost { const double* eps_k; const double* eps_kq; phoebe_elph_rate_params prm; double* rate; };

// one pipelined host batch: copy-in stream -> compute stream -> copy-out stream over staging slot (n mod 2).
// nk_stack > 0: the arrays hold the q lists of nk_stack k slots, k slowest (nq = rows of ALL of them): the stacked forms
int async_batch(phoebe_elph_ctx* c, int32_t nq, int32_t nb2, const double* q_host, const void* Ukq_host,
                const void* ev_host, const double* omega_host, double* out_host, const RateHost* rh, int nk_stack = 0,
                int slot0 = 0)
{
    if (!c->async_ready) {
        PE_CUDA(c, cudaStreamCreateWithFlags(&c->s_in, cudaStreamNonBlocking));
        PE_CUDA(c, cudaStreamCreateWithFlags(&c->s_out, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            PE_CUDA(c, cudaEventCreateWithFlags(&c->ev_in[i], cudaEventDisableTiming));
            PE_CUDA(c, cudaEventCreateWithFlags(&c->ev_done[i], cudaEventDisableTiming));
            PE_CUDA(c, cudaEventCreateWithFlags(&c->ev_out[i], cudaEventDisableTiming));
        }
        c->async_ready = true;
        c->async_n = 0;
    }
    const phoebe_elph_dims& d = c->dims;
    const unsigned slot = c->async_n & 1u;
    const bool reuse = c->async_n >= 2;          // the slot has been used before: order behind its last users
    double* sq = reinterpret_cast<double*>(c->ws + c->L.off_sq + slot * c->L.sz_sq);
    double2* sU = reinterpret_cast<double2*>(c->ws + c->L.off_sUkq + slot * c->L.sz_sUkq);
    double2* sZ = reinterpret_cast<double2*>(c->ws + c->L.off_sev + slot * c->L.sz_sev);
    double* sw = reinterpret_cast<double*>(c->ws + c->L.off_som + slot * c->L.sz_som);
    double* so = reinterpret_cast<double*>(c->ws + c->L.off_sout + slot * c->L.sz_sout);
    // copy-in stream: the compute that last read this input slot must be done
    if (reuse) PE_CUDA(c, cudaStreamWaitEvent(c->s_in, c->ev_done[slot], 0));
    else {      // first use of the slot: order behind whatever the compute stream did with the staging area before
        PE_CUDA(c, cudaEventRecord(c->ev_done[slot], c->stream));
        PE_CUDA(c, cudaStreamWaitEvent(c->s_in, c->ev_done[slot], 0));
    }
    PE_CUDA(c, cudaMemcpyAsync(sq, q_host, (size_t)nq * 24, cudaMemcpyHostToDevice, c->s_in));
    PE_CUDA(c, cudaMemcpyAsync(sU, Ukq_host, (size_t)nq * d.nw * nb2 * 16, cudaMemcpyHostToDevice, c->s_in));
    PE_CUDA(c, cudaMemcpyAsync(sZ, ev_host, (size_t)nq * d.nmodes * d.nmodes * 16, cudaMemcpyHostToDevice, c->s_in));
    PE_CUDA(c, cudaMemcpyAsync(sw, omega_host, (size_t)nq * d.nmodes * 8, cudaMemcpyHostToDevice, c->s_in));
    const size_t nrate = (size_t)std::max(1, nk_stack) * c->nb1;       // rate / eps_k values of this batch
    double* srate = reinterpret_cast<double*>(c->ws + c->L.off_rate) + (size_t)slot * 2 * c->L.nk_slots * d.nb1_max;
    double* se1 = srate + (size_t)c->L.nk_slots * d.nb1_max;
    double* se2 = reinterpret_cast<double*>(c->ws + c->L.off_seps) + (size_t)slot * d.nq_max * d.nb2_max;
    if (rh) {
        // srate is the one buffer both the copy-in and the copy-out stream touch: the copy-out of the batch that last
        // used this slot must have read it before the next initial values land
        if (reuse) PE_CUDA(c, cudaStreamWaitEvent(c->s_in, c->ev_out[slot], 0));
        PE_CUDA(c, cudaMemcpyAsync(srate, rh->rate, nrate * 8, cudaMemcpyHostToDevice, c->s_in));
        PE_CUDA(c, cudaMemcpyAsync(se1, rh->eps_k, nrate * 8, cudaMemcpyHostToDevice, c->s_in));
        PE_CUDA(c, cudaMemcpyAsync(se2, rh->eps_kq, (size_t)nq * nb2 * 8, cudaMemcpyHostToDevice, c->s_in));
    }
    PE_CUDA(c, cudaEventRecord(c->ev_in[slot], c->s_in));
    // compute stream: inputs in, and the copy-out that last read this output slot done
    PE_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_in[slot], 0));
    if (reuse) PE_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_out[slot], 0));
    int rc;
    const int rows_per_k = nk_stack > 0 ? nq / nk_stack : 0;
    if (rh) {
        RateReq rr{se1, se2, rh->prm, srate};
        rc = run_q_batch(c, nq, nb2, sq, sU, sZ, sw, out_host ? so : nullptr, &rr, rows_per_k, slot0);
    } else {
        rc = run_q_batch(c, nq, nb2, sq, sU, sZ, sw, so, nullptr, rows_per_k, slot0);
    }
    if (rc) return rc;
    PE_CUDA(c, cudaEventRecord(c->ev_done[slot], c->stream));
    // copy-out stream
    PE_CUDA(c, cudaStreamWaitEvent(c->s_out, c->ev_done[slot], 0));
    if (rh) PE_CUDA(c, cudaMemcpyAsync(rh->rate, srate, nrate * 8, cudaMemcpyDeviceToHost, c->s_out));
    if (out_host)
        PE_CUDA(c, cudaMemcpyAsync(out_host, so, (size_t)nq * c->nb1 * nb2 * d.nmodes * 8, cudaMemcpyDeviceToHost, c->s_out));
    PE_CUDA(c, cudaEventRecord(c->ev_out[slot], c->s_out));
    c->async_n++;
    return PHOEBE_ELPH_OK;
}
}  // namespace

extern "C" {

int phoebe_elph_q_batch_host_async(phoebe_elph_ctx* c, int32_t nq, int32_t nb2, const double* q_host, const void* Ukq_host,
                                   const void* ev_host, const double* omega_host, double* out_host)
{
    if (!c) return PHOEBE_ELPH_E_NULL;
    if (!c->have_k) return fail(c, PHOEBE_ELPH_E_NO_K, "q_batch_host_async before set_k");
    if (nq == 0) return PHOEBE_ELPH_OK;          // an empty batch is a no-op (nothing is read or written)
    if (!q_host || !Ukq_host || !ev_host || !omega_host || !out_host) return fail(c, PHOEBE_ELPH_E_NULL, "q_batch_host_async: null pointer");
    if (nq < 0 || nq > c->dims.nq_max) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_host_async: nq out of range");
    if (nb2 <= 0 || nb2 > c->dims.nb2_max) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_host_async: nb2 out of range");
    return async_batch(c, nq, nb2, q_host, Ukq_host, ev_host, omega_host, out_host, nullptr);
}

int phoebe_elph_q_batch_rates_host_async(phoebe_elph_ctx* c, int32_t nq, int32_t nb2, const double* q_host,
                                         const void* Ukq_host, const void* ev_host, const double* omega_host,
                                         const double* eps_k_host, const double* eps_kq_host,
                                         const phoebe_elph_rate_params* prm, double* rate_host, double* out_host)
{
    if (!c) return PHOEBE_ELPH_E_NULL;
    if (!c->have_k) return fail(c, PHOEBE_ELPH_E_NO_K, "q_batch_rates_host_async before set_k");
    if (nq == 0) return PHOEBE_ELPH_OK;          // an empty batch is a no-op (nothing is read or written)
    if (!q_host || !Ukq_host || !ev_host || !omega_host || !eps_k_host || !eps_kq_host || !prm || !rate_host)
        return fail(c, PHOEBE_ELPH_E_NULL, "q_batch_rates_host_async: null pointer");
    if (nq < 0 || nq > c->dims.nq_max) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_rates_host_async: nq out of range");
    if (nb2 <= 0 || nb2 > c->dims.nb2_max) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_rates_host_async: nb2 out of range");
    if (!(prm->kT > 0.0) || !(prm->sigma > 0.0)) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_rates_host_async: kT and sigma must be > 0");
    RateHost rh{eps_k_host, eps_kq_host, *prm, rate_host};
    return async_batch(c, nq, nb2, q_host, Ukq_host, ev_host, omega_host, out_host, &rh);
}

namespace {
int check_multi(phoebe_elph_ctx* c, const char* who, int32_t nk, int32_t nq, int32_t nb2)
{
    if (!c->have_k) return fail(c, PHOEBE_ELPH_E_NO_K, "stacked q_batch before set_k_batch");
    if (nk <= 0 || nk > c->nk_have) return fail(c, PHOEBE_ELPH_E_DIMS, "stacked q_batch: nk exceeds the k slots of the last set_k_batch");
    if (nq < 0 || (nq % 64) != 0) return fail(c, PHOEBE_ELPH_E_DIMS, "stacked q_batch: nq must be a multiple of 64");
    if ((long long)nk * nq > c->dims.nq_max) return fail(c, PHOEBE_ELPH_E_DIMS, "stacked q_batch: nk*nq exceeds nq_max");
    if (nb2 <= 0 || nb2 > c->dims.nb2_max) return fail(c, PHOEBE_ELPH_E_DIMS, "stacked q_batch: nb2 out of range");
    if (c->nG > 0) return fail(c, PHOEBE_ELPH_E_DIMS, "stacked q_batch: not available while the polar term is on");
    (void)who;
    return PHOEBE_ELPH_OK;
}
// k slots per pipelined chunk of a stacked host call: the fewest whose stacked rows still fill the GPU for ~8 rounds of
// contraction tiles (a chunk is one contraction launch) -- many small chunks keep the un-overlapped first copy-in and last
// copy-out of a call short (4-atom workload, 16 slots: chunks of 4 -> 1.63 M pairs/s end to end, chunks of 1 -> see bench)
int multi_chunk_slots(const phoebe_elph_ctx* c, int nk, int nq)
{
    const long ntn = ceil_div(c->nb1 * c->dims.nw * c->dims.nmodes, 64);
    const long min_rows = std::max<long>(64, (8L * kSMs + ntn - 1) / ntn * 64);      // rows of ~8 rounds of 64 x 64 tiles
    int kc = 1;
    while (kc < nk && (long)kc * nq < min_rows) ++kc;
    return kc;
}
}  // namespace

int phoebe_elph_q_batch_multi_host_async(phoebe_elph_ctx* c, int32_t nk, int32_t nq, int32_t nb2, const double* q_host,
                                         const void* Ukq_host, const void* ev_host, const double* omega_host, double* out_host)
{
    if (!c) return PHOEBE_ELPH_E_NULL;
    if (!q_host || !Ukq_host || !ev_host || !omega_host || !out_host) return fail(c, PHOEBE_ELPH_E_NULL, "q_batch_multi_host_async: null pointer");
    if (int rc = check_multi(c, "q_batch_multi_host_async", nk, nq, nb2)) return rc;
    if (nq == 0) return PHOEBE_ELPH_OK;
    const phoebe_elph_dims& d = c->dims;
    const int kc = multi_chunk_slots(c, nk, nq);
    for (int j0 = 0; j0 < nk; j0 += kc) {          // chunks of k slots: the copies of one chunk overlap the kernels of its neighbours
        const int nkc = std::min(kc, nk - j0);
        const size_t r0 = (size_t)j0 * nq;
        int rc = async_batch(c, nkc * nq, nb2, q_host + r0 * 3, static_cast<const char*>(Ukq_host) + r0 * d.nw * nb2 * 16,
                             static_cast<const char*>(ev_host) + r0 * d.nmodes * d.nmodes * 16, omega_host + r0 * d.nmodes,
                             out_host + r0 * c->nb1 * nb2 * d.nmodes, nullptr, nkc, j0);
        if (rc) return rc;
    }
    return PHOEBE_ELPH_OK;
}

int phoebe_elph_q_batch_rates_multi_host_async(phoebe_elph_ctx* c, int32_t nk, int32_t nq, int32_t nb2, const double* q_host,
                                               const void* Ukq_host, const void* ev_host, const double* omega_host,
                                               const double* eps_k_host, const double* eps_kq_host,
                                               const phoebe_elph_rate_params* prm, double* rate_host, double* out_host)
{
    if (!c) return PHOEBE_ELPH_E_NULL;
    if (!q_host || !Ukq_host || !ev_host || !omega_host || !eps_k_host || !eps_kq_host || !prm || !rate_host)
        return fail(c, PHOEBE_ELPH_E_NULL, "q_batch_rates_multi_host_async: null pointer");
    if (int rc = check_multi(c, "q_batch_rates_multi_host_async", nk, nq, nb2)) return rc;
    if (!(prm->kT > 0.0) || !(prm->sigma > 0.0)) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_rates_multi_host_async: kT and sigma must be > 0");
    if (nq == 0) return PHOEBE_ELPH_OK;
    const phoebe_elph_dims& d = c->dims;
    const int kc = multi_chunk_slots(c, nk, nq);
    for (int j0 = 0; j0 < nk; j0 += kc) {
        const int nkc = std::min(kc, nk - j0);
        const size_t r0 = (size_t)j0 * nq;
        RateHost rh{eps_k_host + (size_t)j0 * c->nb1, eps_kq_host + r0 * nb2, *prm, rate_host + (size_t)j0 * c->nb1};
        int rc = async_batch(c, nkc * nq, nb2, q_host + r0 * 3, static_cast<const char*>(Ukq_host) + r0 * d.nw * nb2 * 16,
                             static_cast<const char*>(ev_host) + r0 * d.nmodes * d.nmodes * 16, omega_host + r0 * d.nmodes,
                             out_host ? out_host + r0 * c->nb1 * nb2 * d.nmodes : nullptr, &rh, nkc, j0);
        if (rc) return rc;
    }
    return PHOEBE_ELPH_OK;
}

int phoebe_elph_wait(phoebe_elph_ctx* c)
{
    if (!c) return PHOEBE_ELPH_E_NULL;
    PE_CUDA(c, cudaStreamSynchronize(c->stream));
    if (c->async_ready) {
        PE_CUDA(c, cudaStreamSynchronize(c->s_out));
        // later synchronous calls use staging slot 0 on the compute stream: restart the slot bookkeeping
        c->async_n = 0;
    }
    return PHOEBE_ELPH_OK;
}

int phoebe_elph_q_batch_rates(phoebe_elph_ctx* c, int32_t nq, int32_t nb2, const double* q_dev, const void* Ukq_dev,
                              const void* ev_dev, const double* omega_dev, const double* eps_k_dev,
                              const double* eps_kq_dev, const phoebe_elph_rate_params* prm, double* rate_dev,
                              double* out_dev)
{
    if (!c) return PHOEBE_ELPH_E_NULL;
    if (!c->have_k) return fail(c, PHOEBE_ELPH_E_NO_K, "q_batch_rates before set_k");
    if (nq == 0) return PHOEBE_ELPH_OK;          // an empty batch is a no-op (nothing is read or written)
    if (!q_dev || !Ukq_dev || !ev_dev || !omega_dev || !eps_k_dev || !eps_kq_dev || !prm || !rate_dev)
        return fail(c, PHOEBE_ELPH_E_NULL, "q_batch_rates: null pointer");
    if (nq < 0 || nq > c->dims.nq_max) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_rates: nq out of range");
    if (nb2 <= 0 || nb2 > c->dims.nb2_max) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_rates: nb2 out of range");
    if (!(prm->kT > 0.0) || !(prm->sigma > 0.0)) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_rates: kT and sigma must be > 0");
    if (!aligned16(Ukq_dev) || !aligned16(ev_dev)) return fail(c, PHOEBE_ELPH_E_ALIGN, "q_batch_rates: complex input not 16-byte aligned");
    if ((reinterpret_cast<uintptr_t>(q_dev) | reinterpret_cast<uintptr_t>(omega_dev) | reinterpret_cast<uintptr_t>(out_dev) |
         reinterpret_cast<uintptr_t>(eps_k_dev) | reinterpret_cast<uintptr_t>(eps_kq_dev) | reinterpret_cast<uintptr_t>(rate_dev)) & 7u)
        return fail(c, PHOEBE_ELPH_E_ALIGN, "q_batch_rates: double array not 8-byte aligned");
    RateReq rr{eps_k_dev, eps_kq_dev, *prm, rate_dev};
    return run_q_batch(c, nq, nb2, q_dev, static_cast<const double2*>(Ukq_dev), static_cast<const double2*>(ev_dev),
                       omega_dev, out_dev, &rr);
}

int phoebe_elph_q_batch_rates_multi(phoebe_elph_ctx* c, int32_t nk, int32_t nq, int32_t nb2, const double* q_dev,
                                    const void* Ukq_dev, const void* ev_dev, const double* omega_dev, const double* eps_k_dev,
                                    const double* eps_kq_dev, const phoebe_elph_rate_params* prm, double* rate_dev,
                                    double* out_dev)
{
    if (!c) return PHOEBE_ELPH_E_NULL;
    if (!c->have_k) return fail(c, PHOEBE_ELPH_E_NO_K, "q_batch_rates_multi before set_k_batch");
    if (!q_dev || !Ukq_dev || !ev_dev || !omega_dev || !eps_k_dev || !eps_kq_dev || !prm || !rate_dev)
        return fail(c, PHOEBE_ELPH_E_NULL, "q_batch_rates_multi: null pointer");
    if (nk <= 0 || nk > c->nk_have) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_rates_multi: nk exceeds the k slots of the last set_k_batch");
    if (nq < 0 || (nq % 64) != 0) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_rates_multi: nq must be a multiple of 64");
    if (nq == 0) return PHOEBE_ELPH_OK;
    if ((long long)nk * nq > c->dims.nq_max) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_rates_multi: nk*nq exceeds nq_max");
    if (nb2 <= 0 || nb2 > c->dims.nb2_max) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_rates_multi: nb2 out of range");
    if (!(prm->kT > 0.0) || !(prm->sigma > 0.0)) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_rates_multi: kT and sigma must be > 0");
    if (c->nG > 0) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_rates_multi: not available while the polar term is on");
    if (!aligned16(Ukq_dev) || !aligned16(ev_dev)) return fail(c, PHOEBE_ELPH_E_ALIGN, "q_batch_rates_multi: complex input not 16-byte aligned");
    RateReq rr{eps_k_dev, eps_kq_dev, *prm, rate_dev};
    return run_q_batch(c, nk * nq, nb2, q_dev, static_cast<const double2*>(Ukq_dev), static_cast<const double2*>(ev_dev),
                       omega_dev, out_dev, &rr, nq);
}

int phoebe_elph_q_batch_rates_host(phoebe_elph_ctx* c, int32_t nq, int32_t nb2, const double* q_host,
                                   const void* Ukq_host, const void* ev_host, const double* omega_host,
                                   const double* eps_k_host, const double* eps_kq_host,
                                   const phoebe_elph_rate_params* prm, double* rate_host, double* out_host)
{
    if (!c) return PHOEBE_ELPH_E_NULL;
    if (!c->have_k) return fail(c, PHOEBE_ELPH_E_NO_K, "q_batch_rates_host before set_k");
    if (nq == 0) return PHOEBE_ELPH_OK;          // an empty batch is a no-op (nothing is read or written)
    if (!q_host || !Ukq_host || !ev_host || !omega_host || !eps_k_host || !eps_kq_host || !prm || !rate_host)
        return fail(c, PHOEBE_ELPH_E_NULL, "q_batch_rates_host: null pointer");
    if (nq < 0 || nq > c->dims.nq_max) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_rates_host: nq out of range");
    if (nb2 <= 0 || nb2 > c->dims.nb2_max) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_rates_host: nb2 out of range");
    if (!(prm->kT > 0.0) || !(prm->sigma > 0.0)) return fail(c, PHOEBE_ELPH_E_DIMS, "q_batch_rates_host: kT and sigma must be > 0");
    if (int rc0 = drain_async(c)) return rc0;
    const phoebe_elph_dims& d = c->dims;
    double* sq = reinterpret_cast<double*>(c->ws + c->L.off_sq);
    double2* sU = reinterpret_cast<double2*>(c->ws + c->L.off_sUkq);
    double2* sZ = reinterpret_cast<double2*>(c->ws + c->L.off_sev);
    double* sw = reinterpret_cast<double*>(c->ws + c->L.off_som);
    double* so = reinterpret_cast<double*>(c->ws + c->L.off_sout);
    double* srate = reinterpret_cast<double*>(c->ws + c->L.off_rate);
    double* se1 = srate + (size_t)c->L.nk_slots * d.nb1_max;
    double* se2 = reinterpret_cast<double*>(c->ws + c->L.off_seps);
    PE_CUDA(c, cudaMemcpyAsync(sq, q_host, (size_t)nq * 24, cudaMemcpyHostToDevice, c->stream));
    PE_CUDA(c, cudaMemcpyAsync(sU, Ukq_host, (size_t)nq * d.nw * nb2 * 16, cudaMemcpyHostToDevice, c->stream));
    PE_CUDA(c, cudaMemcpyAsync(sZ, ev_host, (size_t)nq * d.nmodes * d.nmodes * 16, cudaMemcpyHostToDevice, c->stream));
    PE_CUDA(c, cudaMemcpyAsync(sw, omega_host, (size_t)nq * d.nmodes * 8, cudaMemcpyHostToDevice, c->stream));
    PE_CUDA(c, cudaMemcpyAsync(srate, rate_host, (size_t)c->nb1 * 8, cudaMemcpyHostToDevice, c->stream));
    PE_CUDA(c, cudaMemcpyAsync(se1, eps_k_host, (size_t)c->nb1 * 8, cudaMemcpyHostToDevice, c->stream));
    PE_CUDA(c, cudaMemcpyAsync(se2, eps_kq_host, (size_t)nq * nb2 * 8, cudaMemcpyHostToDevice, c->stream));
    RateReq rr{se1, se2, *prm, srate};
    int rc = run_q_batch(c, nq, nb2, sq, sU, sZ, sw, out_host ? so : nullptr, &rr);
    if (rc) return rc;
    PE_CUDA(c, cudaMemcpyAsync(rate_host, srate, (size_t)c->nb1 * 8, cudaMemcpyDeviceToHost, c->stream));
    if (out_host)
        PE_CUDA(c, cudaMemcpyAsync(out_host, so, (size_t)nq * c->nb1 * nb2 * d.nmodes * 8, cudaMemcpyDeviceToHost, c->stream));
    PE_CUDA(c, cudaStreamSynchronize(c->stream));
    return PHOEBE_ELPH_OK;
}

int phoebe_elph_copy_g1(phoebe_elph_ctx* c, void* dst_dev, size_t dst_bytes)
{
    if (!c) return PHOEBE_ELPH_E_NULL;
    if (!dst_dev) return fail(c, PHOEBE_ELPH_E_NULL, "copy_g1: null pointer");
    if (!c->have_k) return fail(c, PHOEBE_ELPH_E_NO_K, "copy_g1 before set_k");
    const size_t bytes = (size_t)c->dims.nRp * c->nb1 * c->dims.nw * c->dims.nmodes * 16;
    if (dst_bytes < bytes) return fail(c, PHOEBE_ELPH_E_WORKSPACE, "copy_g1: destination too small");
    PE_CUDA(c, cudaMemcpyAsync(dst_dev, c->g1, bytes, cudaMemcpyDeviceToDevice, c->stream));
    return PHOEBE_ELPH_OK;
}

int phoebe_elph_set_polar(phoebe_elph_ctx* c, const double* recip_host, int32_t nG, const double* G_host,
                          const double* Zstar_host, const double* eps_inf_host, double coeff)
{
    if (!c) return PHOEBE_ELPH_E_NULL;
    if (nG == 0) { c->nG = 0; return PHOEBE_ELPH_OK; }
    if (!recip_host || !G_host || !Zstar_host || !eps_inf_host) return fail(c, PHOEBE_ELPH_E_NULL, "set_polar: null pointer");
    if (nG < 0 || nG > kMaxG) return fail(c, PHOEBE_ELPH_E_DIMS, "set_polar: nG out of range (<= 4096)");
    if (c->dims.nmodes % 3) return fail(c, PHOEBE_ELPH_E_DIMS, "set_polar: nmodes is not 3 x atoms");
    if (c->phase_sign != 1.0 || c->conj_Uk || !c->conj_Ukq || c->conj_ev)
        return fail(c, PHOEBE_ELPH_E_DIMS, "set_polar: the polar term belongs to the el-ph conventions");
    PE_CUDA(c, cudaMemcpyAsync(c->ws + c->L.off_G, G_host, (size_t)nG * 24, cudaMemcpyHostToDevice, c->stream));
    PE_CUDA(c, cudaMemcpyAsync(c->ws + c->L.off_Zstar, Zstar_host, (size_t)(c->dims.nmodes / 3) * 72, cudaMemcpyHostToDevice, c->stream));
    PE_CUDA(c, cudaStreamSynchronize(c->stream));      // the host arrays may be pageable
    for (int i = 0; i < 9; ++i) { c->polar.recip[i] = recip_host[i]; c->polar.eps[i] = eps_inf_host[i]; }
    c->polar.coeff = coeff;
    c->nG = nG;
    return PHOEBE_ELPH_OK;
}

int phoebe_elph_set_conventions(phoebe_elph_ctx* c, int32_t phase_sign, int32_t conj_Uk, int32_t conj_Ukq, int32_t conj_ev)
{
    if (!c) return PHOEBE_ELPH_E_NULL;
    if (phase_sign != 1 && phase_sign != -1) return fail(c, PHOEBE_ELPH_E_DIMS, "set_conventions: phase_sign must be +1 or -1");
    const bool dflt = phase_sign == 1 && !conj_Uk && conj_Ukq && !conj_ev;
    if (!dflt && c->nG > 0) return fail(c, PHOEBE_ELPH_E_DIMS, "set_conventions: the polar term belongs to the el-ph conventions");
    c->phase_sign = (double)phase_sign;
    c->conj_Uk = conj_Uk != 0; c->conj_Ukq = conj_Ukq != 0; c->conj_ev = conj_ev != 0;
    c->have_k = false;                  // a g1' computed under other conventions must not be reused
    return PHOEBE_ELPH_OK;
}

int phoebe_elph_g1_buffer(phoebe_elph_ctx* c, int32_t slot, void** ptr_out, size_t* bytes_out, size_t* stride_out)
{
    if (!c) return PHOEBE_ELPH_E_NULL;
    if (!ptr_out || !bytes_out) return fail(c, PHOEBE_ELPH_E_NULL, "g1_buffer: null pointer");
    if (!c->have_k) return fail(c, PHOEBE_ELPH_E_NO_K, "g1_buffer before set_k");
    if (slot < -1 || slot >= c->nk_have) return fail(c, PHOEBE_ELPH_E_DIMS, "g1_buffer: slot out of range");
    const size_t one = (size_t)c->dims.nRp * c->nb1 * c->dims.nw * c->dims.nmodes * 16;
    const size_t stride = c->L.g1_stride * 16;
    c->g1P_stale = true;                 // the caller may change g1' in place (Re-pool all-reduce): re-pack before the next a4
    c->Bi8_stale = true;
    if (stride_out) *stride_out = stride;
    if (slot >= 0) {
        *ptr_out = c->g1_base + (size_t)slot * c->L.g1_stride;
        *bytes_out = one;
    } else {
        *ptr_out = c->g1_base;
        *bytes_out = (size_t)(c->nk_have - 1) * stride + one;
    }
    return PHOEBE_ELPH_OK;
}

int phoebe_elph_launch_counts(const phoebe_elph_ctx* c, int64_t* counts)
{
    if (!c || !counts) return PHOEBE_ELPH_E_NULL;
    for (int i = 0; i < PHOEBE_ELPH_K_COUNT; ++i) counts[i] = c->launches[i];
    return PHOEBE_ELPH_OK;
}

int phoebe_elph_profile(phoebe_elph_ctx* c, int32_t enable)
{
    if (!c) return PHOEBE_ELPH_E_NULL;
    c->prof = enable != 0;
    return PHOEBE_ELPH_OK;
}

int phoebe_elph_profile_read(phoebe_elph_ctx* c, double* ms, int64_t* launches)
{
    if (!c || !ms || !launches) return PHOEBE_ELPH_E_NULL;
    PE_CUDA(c, cudaStreamSynchronize(c->stream));
    for (int i = 0; i < PHOEBE_ELPH_K_COUNT; ++i) { ms[i] = 0.0; launches[i] = 0; }
    for (const EventPair& p : c->evs) {
        float t = 0.f;
        PE_CUDA(c, cudaEventElapsedTime(&t, p.a, p.b));
        ms[p.kind] += t;
        launches[p.kind]++;
        c->ev_pool.push_back(p.a);
        c->ev_pool.push_back(p.b);
    }
    c->evs.clear();
    return PHOEBE_ELPH_OK;
}

int phoebe_elph_set_tuning(phoebe_elph_ctx* c, const char* key, int64_t value)
{
    if (!c || !key) return PHOEBE_ELPH_E_NULL;
    if (!strcmp(key, "nq_sub")) {
        if (value < 1) return fail(c, PHOEBE_ELPH_E_DIMS, "nq_sub must be >= 1");
        // a multiple of the phase padding (128): sub-batch offsets then never split a contraction row tile (stacked
        // forms: a tile must not straddle two k slots)
        c->nq_sub = (int)std::min<int64_t>(std::max<int64_t>(kQPad, value / kQPad * kQPad), c->L.nq_sub);
        return PHOEBE_ELPH_OK;
    }
    if (!strcmp(key, "tile")) {
        if (value != 0 && value != 32 && value != 64)
            return fail(c, PHOEBE_ELPH_E_DIMS, "tile must be 0, 32 or 64");
        c->tile = (int)value;
        return PHOEBE_ELPH_OK;
    }
    if (!strcmp(key, "m3")) { c->m3 = value != 0; return PHOEBE_ELPH_OK; }
    if (!strcmp(key, "planar")) { c->planar = value != 0; return PHOEBE_ELPH_OK; }
    if (!strcmp(key, "pair_ctas")) {
        if (value < 1 || value > 2) return fail(c, PHOEBE_ELPH_E_DIMS, "pair_ctas must be 1 or 2");
        c->pair_ctas = (int)value;
        return PHOEBE_ELPH_OK;
    }
    if (!strcmp(key, "pair")) {
        if (value < 0 || value > 2) return fail(c, PHOEBE_ELPH_E_DIMS, "pair must be 0, 1 or 2");
        c->pair = (int)value;
        c->last_pair = -1;
        return PHOEBE_ELPH_OK;
    }
    if (!strcmp(key, "rot_plain")) { c->rot_plain = value != 0; return PHOEBE_ELPH_OK; }
    if (!strcmp(key, "qfold")) { c->qfold = value != 0; return PHOEBE_ELPH_OK; }
    if (!strcmp(key, "i8")) { c->i8 = value != 0 ? 1 : 0; return PHOEBE_ELPH_OK; }
    if (!strcmp(key, "i8_cluster")) { c->i8_cluster = (value == 1 || value == 2 || value == 4 || value == 8) ? value : 0; return PHOEBE_ELPH_OK; }
    if (!strcmp(key, "setk_pair")) { c->setk_pair = value != 0; return PHOEBE_ELPH_OK; }
    if (!strcmp(key, "rot_blk")) {
        if (value < 0 || value > 2) return fail(c, PHOEBE_ELPH_E_DIMS, "rot_blk must be 0, 1 or 2");
        c->rot_blk = (int)value;
        return PHOEBE_ELPH_OK;
    }
    if (!strcmp(key, "rot_qg") || !strcmp(key, "rot_gb1") || !strcmp(key, "rot_mtw")) {
        if (value < 0 || value > 1024) return fail(c, PHOEBE_ELPH_E_DIMS, "rotation geometry override out of range");
        (key[4] == 'q' ? c->rot_qg : key[4] == 'g' ? c->rot_gb1 : c->rot_mtw) = (int)value;
        return PHOEBE_ELPH_OK;
    }
    if (!strcmp(key, "s_split")) {
        if (value < 0 || value > c->L.S_alloc) return fail(c, PHOEBE_ELPH_E_DIMS, "s_split out of range");
        c->s_split = (int)value;
        return PHOEBE_ELPH_OK;
    }
    return fail(c, PHOEBE_ELPH_E_DIMS, "unknown tuning key");
}

int phoebe_elph_get_tuning(const phoebe_elph_ctx* c, const char* key, int64_t* value)
{
    if (!c || !key || !value) return PHOEBE_ELPH_E_NULL;
    if (!strcmp(key, "nq_sub")) { *value = c->nq_sub; return PHOEBE_ELPH_OK; }
    if (!strcmp(key, "m3")) { *value = c->m3 ? 1 : 0; return PHOEBE_ELPH_OK; }
    // real rows of the +R / -R pair form if the LAST contraction launch used it, else 0 (before any launch: whether the
    // 64 x 64 tile would use it with the current knobs)
    if (!strcmp(key, "pair_rows")) {
        const bool on = c->m3 && c->planar && (c->tile == 0 || c->tile == 64) && c->pair_Kr > 0 &&
                        (c->pair == 2 || (c->pair == 1 && (size_t)4 * c->pair_Kr < (size_t)6 * c->dims.nRp));
        *value = (c->last_pair < 0 ? on : c->last_pair == 1) ? c->pair_Kr : 0;
        return PHOEBE_ELPH_OK;
    }
    if (!strcmp(key, "s_split")) {
        *value = c->s_split > 0 ? c->s_split
                                : setk_auto_split(c->dims.nRe, c->dims.nRp, c->dims.nw * c->dims.nw * c->dims.nmodes);
        return PHOEBE_ELPH_OK;
    }
    if (!strcmp(key, "s_alloc")) { *value = c->L.S_alloc; return PHOEBE_ELPH_OK; }
    if (!strcmp(key, "i8")) { *value = c->last_i8 < 0 ? c->i8 : c->last_i8; return PHOEBE_ELPH_OK; }
    if (!strcmp(key, "i8_cluster")) { *value = c->last_i8_cluster ? c->last_i8_cluster : c->i8_cluster; return PHOEBE_ELPH_OK; }
    if (!strcmp(key, "i8_grid")) { *value = c->last_i8_grid; return PHOEBE_ELPH_OK; }      // CTAs of the last INT8 contraction launch   // did the last a4 run on INT8
    // ring rows of the a1 pair form (2 per +R / -R pair of the Re list) if the LAST set_k_batch used it, else 0
    if (!strcmp(key, "setk_pair_rows")) { *value = c->last_setk_pair ? 2 * c->npairE : 0; return PHOEBE_ELPH_OK; }
    if (!strcmp(key, "qfold_reps")) {       // representatives of the last q_batch call if it took the fold, else 0
        *value = 0;
        if (c->last_fold) {
            int meta[2] = {0, 0};
            if (cudaMemcpyAsync(meta, c->ws + c->L.off_fold, 8, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess ||
                cudaStreamSynchronize(c->stream) != cudaSuccess) return PHOEBE_ELPH_E_CUDA;
            *value = meta[1] ? meta[0] : 0;
        }
        return PHOEBE_ELPH_OK;
    }
    if (!strcmp(key, "nq_sub_max")) { *value = c->L.nq_sub; return PHOEBE_ELPH_OK; }
    // byte offsets of the C and Pt scratch areas inside the workspace (debugging aids for the tests)
    if (!strcmp(key, "off_C")) { *value = (int64_t)c->L.off_C; return PHOEBE_ELPH_OK; }
    if (!strcmp(key, "off_Pt")) { *value = (int64_t)c->L.off_Pt; return PHOEBE_ELPH_OK; }
    if (!strcmp(key, "ldq")) { *value = c->L.ldq; return PHOEBE_ELPH_OK; }
    return PHOEBE_ELPH_E_DIMS;
}

int phoebe_elph_destroy(phoebe_elph_ctx* c)
{
    if (!c) return PHOEBE_ELPH_E_NULL;
    for (const EventPair& p : c->evs) { cudaEventDestroy(p.a); cudaEventDestroy(p.b); }
    for (cudaEvent_t e : c->ev_pool) cudaEventDestroy(e);
    if (c->async_ready) {
        for (int i = 0; i < 2; ++i) { cudaEventDestroy(c->ev_in[i]); cudaEventDestroy(c->ev_done[i]); cudaEventDestroy(c->ev_out[i]); }
        cudaStreamDestroy(c->s_in); cudaStreamDestroy(c->s_out);
    }
    delete c;
    return PHOEBE_ELPH_OK;
}

const char* phoebe_elph_last_error(const phoebe_elph_ctx* c) { return c ? c->err.c_str() : ""; }

}  // extern "C"
