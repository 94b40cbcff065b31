// rfa_api.cpp -- host logic and the C ABI of librfa.so (include/rfa.h).
//
// Host side of the hot path: validation, the per-label coefficient table in fp64 (rounded once to
// fp32), the monotone stability check, workspace layout, the plan of the temporally blocked kernel,
// ping-pong bookkeeping (Alg. 2).  All device work goes through the launchers of
// rfa_kernels.cu on the caller's stream.  There is no CPU fallback: without a CUDA device rfa_create
// fails with RFA_E_CUDA.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/rfa.h"
#include "rfa_internal.h"

static thread_local std::string g_err;

static int fail(int code, const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_err = buf;
    return code;
}

static int cuda_fail(cudaError_t e, const char *what)
{
    return fail(RFA_E_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

struct rfa_sim {
    RfaGrid g{};
    size_t nvox = 0;
    double h_m[3]{};                     // spacing in metres
    double dt = 0, t_blood = 0;
    std::vector<rfa_tissue> table;
    uint32_t label_held_mask = 0;
    std::vector<double> q_power;         // per scenario, W/m^3 (0 unless a POWER needle is set)
    cudaStream_t stream = nullptr;
    unsigned char *ws = nullptr;         // device workspace
    bool own_ws = false;
    float *theta[2]{};                   // ping-pong temperature images (theta = T - T_a)
    unsigned char *resid[2]{};           // ping-pong fp16 residual images (rfa_device.cuh: rfa_advance)
    int cur = 0;                         // index of the current image
    uint8_t *state = nullptr;            // packed state bytes
    float *tables = nullptr;             // batch x 3 x 128 coefficients
    float *kap = nullptr;                // 16 x 16 face factors Kf/K_c - 1 (conservative conduction, R-28)
    int conduction = RFA_COND_EQ12;
    unsigned char *scratch = nullptr;    // nvox*4 bytes staging
    unsigned long long *counters = nullptr;
    int kernel = RFA_KERNEL_AUTO;
    int fused = 3;
    RfaTbPlan plans_by_mode[2][5]{};     // [conduction mode][fused steps 1..4]: the conservative variant needs more
    int resident[2][5][RFA_N_SHAPES]{};  // shared memory (deeper state ring), so its occupancy and plan may differ
    const RfaTbPlan *plans() const { return plans_by_mode[conduction == RFA_COND_FACE ? 1 : 0]; }
    long long launches = 0;
    long long *probes = nullptr;         // device, n_probes flat voxel indices (library-owned)
    int n_probes = 0;
    float *record = nullptr;             // device staging of rfa_step_record (library-owned, grows on demand)
    size_t record_cap = 0;               // floats
    float *stage = nullptr;              // device staging of host displacement fields / host images (library-owned,
    size_t stage_cap = 0;                // grows on demand; floats)
    RfaTensorMap tm_theta[2]{};          // tensor maps of the two temperature images and of the state volume (TMA-staged
    RfaTensorMap tm_state{};             // one-step kernel, rfa_stream.cu)
    bool stream_ok = false;              // the grid has a TMA path (nx % 16 == 0, driver entry point found)
    RfaTbPlan stream_plan{};
    unsigned long long stream_draws = 0; // items drawn so far from the dynamic work counter (counters[4]; never reset)
    RfaTensorMap tm_blk_theta[2][RFA_N_SHAPES]{};   // blocked kernel, TMA variant: maps of the two images / the state volume
    RfaTensorMap tm_blk_state[RFA_N_SHAPES]{};      // per tile shape
    // Residual-prefetch variant of the blocked kernel (rfa_kernels.cu: RPF): chosen from the share of warp-planes that took
    // the compensated path, which the kernels count in counters[5]; the count is read back without ever waiting for the
    // stream (an 8-byte copy into pinned memory + an event that later launches poll)
    int res_prefetch_mode = RFA_RES_PREFETCH_AUTO;
    int res_prefetch_on = 0;
    unsigned long long *hot_host = nullptr;   // pinned
    cudaEvent_t hot_evt = nullptr;
    bool hot_pending = false;
    unsigned long long hot_seen = 0;          // counter value at the last completed sample
    double planes_issued = 0, planes_at_sample = 0, planes_seen = 0;   // warp-planes launched: now / at the pending sample / at the last completed one
    double hot_fraction = 0;                  // last completed sample
    int launches_since_sample = 0;
    int staging = RFA_STAGING_AUTO;      // rfa_configure_staging
    int force_shape = -1;                // rfa_configure_tile: -1 = the planner chooses
    int device = 0;                      // the CUDA device the simulation lives on (current device at rfa_create)
    int held_copy_auto = 0;              // what rfa_create chose for the held-copy variant (RFA_HELD_COPY_AUTO)
};

// Every entry point that touches the device runs on the simulation's own device, whatever the caller's current
// device is, and puts the caller's device back on return.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(const rfa_sim *s)
    {
        if (s && cudaGetDevice(&prev) == cudaSuccess && prev != s->device) switched = cudaSetDevice(s->device) == cudaSuccess;
    }
    ~DeviceGuard()
    {
        if (switched) cudaSetDevice(prev);
    }
};

// library-owned device staging buffer of at least `floats` floats (the stream is drained before it is replaced)
static int ensure_stage(rfa_sim *s, size_t floats)
{
    if (s->stage_cap >= floats) return RFA_OK;
    cudaError_t e = cudaStreamSynchronize(s->stream);
    if (e != cudaSuccess) return RFA_E_CUDA;
    if (s->stage) cudaFree(s->stage);
    s->stage = nullptr;
    s->stage_cap = 0;
    e = cudaMalloc((void **)&s->stage, floats * sizeof(float));
    if (e != cudaSuccess) {
        cudaGetLastError();
        return RFA_E_NOMEM;
    }
    s->stage_cap = floats;
    return RFA_OK;
}

// ------------------------------------------------------------------------------------------------
// workspace layout
// ------------------------------------------------------------------------------------------------
static size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

struct WsLayout {
    size_t theta0, theta1, resid0, resid1, state, tables, kap, scratch, counters, total;
};

static bool ws_layout(const int dims[3], int batch, WsLayout &L)
{
    if (!dims || batch < 1) return false;
    for (int a = 0; a < 3; ++a)
        if (dims[a] < 1 || (a > 0 && dims[a] > 65535)) return false;   // ny, nz are grid dimensions of the set-up kernels
    const double nv = (double)dims[0] * dims[1] * dims[2];
    if (nv * batch > 1.0e11) return false;
    const size_t nvox = (size_t)dims[0] * dims[1] * dims[2];
    size_t off = 0;
    L.theta0 = off;
    off = align256(off + nvox * batch * 4);
    L.theta1 = off;
    off = align256(off + nvox * batch * 4);
    L.resid0 = off;
    off = align256(off + nvox * batch * 2);
    L.resid1 = off;
    off = align256(off + nvox * batch * 2);
    L.state = off;
    off = align256(off + nvox * batch);
    L.tables = off;
    off = align256(off + (size_t)batch * 3 * RFA_TABLE_N * 4);
    L.kap = off;
    off = align256(off + RFA_NLABEL * RFA_NLABEL * 4);
    L.scratch = off;
    off = align256(off + nvox * 4);
    L.counters = off;
    off = align256(off + 256 + 256 * 8);                     // 32 counters + the 256 bins of the label histogram
    L.total = off;
    return true;
}

extern "C" size_t rfa_workspace_bytes(const int dims[3], int batch)
{
    WsLayout L;
    return ws_layout(dims, batch, L) ? L.total : 0;
}

// ------------------------------------------------------------------------------------------------
// host numerics
// ------------------------------------------------------------------------------------------------
static bool tissue_ok(const rfa_tissue &t)
{
    if (!std::isfinite(t.k) || !std::isfinite(t.rho) || !std::isfinite(t.cp) || !std::isfinite(t.wb_cb) ||
        !std::isfinite(t.q_m) || !std::isfinite(t.t_init))
        return false;
    if (t.flags & RFA_TISSUE_HELD) return true;
    return t.k > 0.f && t.rho > 0.f && t.cp > 0.f && t.wb_cb >= 0.f;
}

extern "C" double rfa_stability_number(const float spacing_mm[3], const rfa_tissue *table, int n_tissue, float dt_s)
{
    if (!spacing_mm || !table || n_tissue < 1 || !(dt_s > 0.f)) return -1.0;
    double w = 0;
    for (int a = 0; a < 3; ++a) {
        if (!(spacing_mm[a] > 0.f) || !std::isfinite(spacing_mm[a])) return -1.0;
        const double h = (double)spacing_mm[a] * 1.0e-3;
        w += 1.0 / (h * h);
    }
    double worst = 0;
    for (int l = 0; l < n_tissue; ++l) {
        const rfa_tissue &t = table[l];
        if (!tissue_ok(t)) return -1.0;
        if (t.flags & RFA_TISSUE_HELD) continue;
        const double rc = (double)t.rho * t.cp;
        worst = std::max(worst, (double)dt_s * (2.0 * (double)t.k / rc * w + (double)t.wb_cb / rc));
    }
    return worst;
}

// coefficient table of one scenario (see rfa_device.cuh); fp64, rounded once
static void build_table(const rfa_sim *s, double q_power, RfaTableHost &out)
{
    const double W = 1.0 / (s->h_m[0] * s->h_m[0]) + 1.0 / (s->h_m[1] * s->h_m[1]) + 1.0 / (s->h_m[2] * s->h_m[2]);
    for (int e = 0; e < RFA_TABLE_N; ++e) {
        const int l = e & (int)RFA_ST_LABEL;
        const bool dir = (e & (int)RFA_ST_DIRICHLET) != 0;
        const bool pow = (e & (int)RFA_ST_POWER) != 0;
        double a = 0, nk = 0, qa = 0;
        if (l < (int)s->table.size() && !dir && !(s->table[l].flags & RFA_TISSUE_HELD)) {
            const rfa_tissue &t = s->table[l];
            const double kw = (double)t.k * W;
            a = s->dt / ((double)t.rho * t.cp) * kw;
            nk = -(double)t.wb_cb / kw;
            qa = ((double)t.q_m + (pow ? q_power : 0.0)) / kw;
        }
        out.a[e] = (float)a;
        out.np[e] = (float)nk;
        out.qa[e] = (float)qa;
    }
}

// ------------------------------------------------------------------------------------------------
// plan of the blocked kernel (host only)
// ------------------------------------------------------------------------------------------------
static RfaTbPlan plan_shape(int nx, int ny, int nz, int batch, int S, int shape, int resident_ctas, int tma, double &cost_out)
{
    RfaTbPlan p{};
    p.fused = S;
    p.shape = shape;
    p.tma = tma;
    cost_out = 1e300;
    if (resident_ctas < 1) return p;
    const int RY = RFA_TB_SHAPE[shape][S].ry;
    const int BX = 4 * RFA_TB_SHAPE[shape][S].tx, BY = RY * RFA_TB_SHAPE[shape][S].ty;
    if (BY <= 2 * S) return p;
    // TMA-staged variant: Eq. 12 kernels with 2 or 3 fused steps, state rows of a multiple of 16 bytes, whole thread rows
    if (tma && (S < 2 || S > 3 || (nx % 16) != 0 || (ny % RY) != 0)) return p;
    // its first tile starts SR = S rounded up to a multiple of RY rows above the grid (rfa_kernels.cu), SR - S more than needed
    const int lead = tma ? (S + RY - 1) / RY * RY - S : 0;
    p.tiles_x = nx <= BX ? 1 : (nx - 8 + (BX - 8) - 1) / (BX - 8);
    p.tiles_y = (ny + lead + (BY - 2 * S) - 1) / (BY - 2 * S);
    const long long per_z = (long long)p.tiles_x * p.tiles_y * batch;
    // choose the number of z chunks: minimise rounds * (planes streamed per item + fixed cost)
    double best = 1e300;
    for (int nzc = 1; nzc <= nz; ++nzc) {
        const int zchunk = (nz + nzc - 1) / nzc;
        if ((nzc - 1) * zchunk >= nz) continue;              // empty last chunk
        const long long items = per_z * nzc;
        const long long rounds = (items + resident_ctas - 1) / resident_ctas;
        const double cost = (double)rounds * (zchunk + 2 * S + 3);
        if (cost < best - 1e-9) {
            best = cost;
            p.nzc = nzc;
            p.zchunk = zchunk;
        }
    }
    const long long items = per_z * p.nzc;
    if (items > 0x7fffffffLL) return p;
    p.n_items = (int)items;
    p.grid = (int)std::min<long long>(items, resident_ctas);
    p.ok = 1;
    cost_out = best;
    return p;
}

RfaTbPlan rfa_plan_blocked(int nx, int ny, int nz, int batch, int fused, const int resident_ctas[RFA_N_SHAPES], int tma)
{
    RfaTbPlan best{};
    best.fused = fused;
    best.tma = tma;
    const int S = fused;
    if (S < 1 || S > 4 || nx < 4 || (nx % 4) != 0 || ny < S || nz < S || batch < 1 || !resident_ctas) return best;
    // the kernel addresses one scenario with 32-bit float4 offsets; larger volumes take the plain kernel
    if ((long long)(nx / 4) * ny * nz >= 0x7fffffffLL || (long long)nz * batch >= 0x7fffffffLL) return best;
    double best_cost = 1e300;
    for (int shape = 0; shape < RFA_N_SHAPES; ++shape) {
        double cost;
        RfaTbPlan p = plan_shape(nx, ny, nz, batch, S, shape, resident_ctas[shape], tma, cost);
        // every CTA has 256 threads and 8 voxels per thread and plane, so plane iterations compare directly;
        // the wide shape must win by 5 % (its y halo costs more redundant rows per useful one)
        if (p.ok && cost < best_cost * (shape == 0 ? 1.0 : 0.95)) {
            best = p;
            best_cost = cost;
        }
    }
    return best;
}

// Plan of the TMA-staged one-step kernel: 128 x 16 tiles without redundant voxels (the halo is loaded, not computed).  The
// work items (tile x z chunk) are handed out dynamically, so the chunk length trades the two neighbour planes every
// chunk streams on top of its own against the tail of the last round: cost = planes per CTA + one item (measured on the
// B200, C4: 8 / 12 / 16 / 22 / 32 chunks -> 114 / 111 / 109 / 113 / 119 us per step).
RfaTbPlan rfa_plan_stream(int nx, int ny, int nz, int batch, int resident_ctas)
{
    RfaTbPlan p{};
    p.fused = 1;
    if (resident_ctas < 1 || nx < 1 || ny < 1 || nz < 1 || batch < 1 || (nx % 16) != 0) return p;
    if ((long long)(nx / 4) * ny * nz >= 0x7fffffffLL) return p;
    p.tiles_x = (nx + RFA_STREAM_BX - 1) / RFA_STREAM_BX;
    p.tiles_y = (ny + RFA_STREAM_BY - 1) / RFA_STREAM_BY;
    const long long per_z = (long long)p.tiles_x * p.tiles_y * batch;
    double best = 1e300;
    for (int nzc = 1; nzc <= nz; ++nzc) {
        const int zchunk = (nz + nzc - 1) / nzc;
        if ((nzc - 1) * zchunk >= nz) continue;
        const long long items = per_z * nzc;
        const double item_planes = zchunk + 3;                   // two neighbour planes + pipeline refill
        const double cost = (double)items * item_planes / resident_ctas + item_planes;
        if (cost < best - 1e-9) {
            best = cost;
            p.nzc = nzc;
            p.zchunk = zchunk;
        }
    }
    const long long items = per_z * p.nzc;
    if (p.nzc < 1 || items > 0x7fffffffLL) return p;
    p.n_items = (int)items;
    p.grid = (int)std::min<long long>(items, resident_ctas);
    p.ok = 1;
    return p;
}

// exported for the CPU unit tests of the planner (no GPU needed)
extern "C" int rfa_plan_query(const int dims[3], int batch, int fused, int resident_ctas, int staging, int out[9])
{
    if (!dims || !out) return RFA_E_INVALID;
    if (staging != RFA_STAGING_CP_ASYNC && staging != RFA_STAGING_TMA) return RFA_E_INVALID;
    const int res[RFA_N_SHAPES] = {resident_ctas, resident_ctas};
    RfaTbPlan p = rfa_plan_blocked(dims[0], dims[1], dims[2], batch, fused, res, staging == RFA_STAGING_TMA ? 1 : 0);
    out[0] = p.ok;
    out[1] = p.tiles_x;
    out[2] = p.tiles_y;
    out[3] = p.nzc;
    out[4] = p.zchunk;
    out[5] = p.n_items;
    out[6] = p.grid;
    out[7] = p.ok ? 4 * RFA_TB_SHAPE[p.shape][fused].tx : 0;
    out[8] = p.ok ? RFA_TB_SHAPE[p.shape][fused].ry * RFA_TB_SHAPE[p.shape][fused].ty : 0;
    return RFA_OK;
}

// ------------------------------------------------------------------------------------------------
// helpers
// ------------------------------------------------------------------------------------------------
static bool is_device_ptr(const void *p)
{
    cudaPointerAttributes at{};
    cudaError_t e = cudaPointerGetAttributes(&at, p);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

static int check_sim(rfa_sim *s, int scenario)
{
    if (!s) return fail(RFA_E_INVALID, "null simulation handle");
    if (scenario < 0 || scenario >= s->g.batch) return fail(RFA_E_INVALID, "scenario %d out of range [0,%d)", scenario, s->g.batch);
    return RFA_OK;
}

static int upload_table(rfa_sim *s, int scenario)
{
    RfaTableHost t;
    build_table(s, s->q_power[scenario], t);
    cudaError_t e = rfa_launch_table(t, s->tables + (size_t)scenario * 3 * RFA_TABLE_N, s->stream);
    s->launches++;
    if (e != cudaSuccess) return cuda_fail(e, "table upload");
    return RFA_OK;
}

// Default number of fused steps: 3, except where the planner chose the 128 x 16 tile, whose y halo makes the third
// level expensive (10 useful rows of 16 at S = 3, 12 at S = 2; measured on the 128^3 volumes: 696 vs 670 GVox/s).
static int default_fused(const rfa_sim *s)
{
    if (s->plans()[3].ok && s->plans()[3].shape == 1 && s->plans()[2].ok) return 2;
    return 3;
}

static void make_plans(rfa_sim *s)
{
    s->stream_ok = rfa_stream_make_maps(s->g, s->theta[0], s->state, &s->tm_theta[0], &s->tm_state) &&
                   rfa_stream_make_maps(s->g, s->theta[1], nullptr, &s->tm_theta[1], nullptr);
    s->stream_plan = s->stream_ok ? rfa_plan_stream(s->g.nx, s->g.ny, s->g.nz, s->g.batch, rfa_stream_resident_ctas()) : RfaTbPlan{};
    if (!s->stream_plan.ok) s->stream_ok = false;
    // tensor maps of the blocked kernel's TMA variant: box = the tile of each shape (the same for 2 and 3 fused steps)
    bool blk_maps[RFA_N_SHAPES];
    for (int sh = 0; sh < RFA_N_SHAPES; ++sh) {
        int bx = 0, by = 0, bx3 = 0, by3 = 0;
        rfa_blocked_tile(2, sh, &bx, &by);
        rfa_blocked_tile(3, sh, &bx3, &by3);
        blk_maps[sh] = bx == bx3 && by == by3 && rfa_make_tile_map(s->g, s->theta[0], 4, bx, by, &s->tm_blk_theta[0][sh]) &&
                       rfa_make_tile_map(s->g, s->theta[1], 4, bx, by, &s->tm_blk_theta[1][sh]) &&
                       rfa_make_tile_map(s->g, s->state, 1, bx + 16, by, &s->tm_blk_state[sh]);
    }
    for (int f = 1; f <= 4; ++f) {
        for (int m = 0; m < 2; ++m) {
            int res_tma[RFA_N_SHAPES];
            for (int sh = 0; sh < RFA_N_SHAPES; ++sh) {
                const bool want = s->force_shape < 0 || s->force_shape == sh;
                s->resident[m][f][sh] = want ? rfa_blocked_resident_ctas(f, sh, m, 0) : 0;
                res_tma[sh] = (want && m == 0 && blk_maps[sh] && s->staging != RFA_STAGING_CP_ASYNC) ? rfa_blocked_resident_ctas(f, sh, m, 1) : 0;
            }
            // AUTO: the TMA-staged variant where it measured faster on the B200 -- the 128 x 16 tile (C5: 684 -> 704 GVox/s);
            // with the 64 x 32 tile it executes more instructions than it saves (row-major state tile: two 4-byte loads per
            // level instead of one 8-byte load, more index arithmetic) and the per-thread cp.async variant wins
            // (C4: 783 vs 707), profiles/r2_blocked_ab_ncu.md
            const RfaTbPlan pc = rfa_plan_blocked(s->g.nx, s->g.ny, s->g.nz, s->g.batch, f, s->resident[m][f], 0);
            const RfaTbPlan pt = rfa_plan_blocked(s->g.nx, s->g.ny, s->g.nz, s->g.batch, f, res_tma, 1);
            const bool take_tma = pt.ok && (s->staging == RFA_STAGING_TMA || !pc.ok || (pt.shape == 1 && pc.shape == 1));
            s->plans_by_mode[m][f] = take_tma ? pt : pc;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// C ABI
// ------------------------------------------------------------------------------------------------
extern "C" const char *rfa_last_error(void) { return g_err.c_str(); }

extern "C" int rfa_create(rfa_sim **out, const int dims[3], const float spacing_mm[3], const uint8_t *labels,
                          const rfa_tissue *table, int n_tissue, float t_blood_c, float dt_s, int batch,
                          void *workspace, size_t workspace_bytes, void *cuda_stream)
{
    if (!out) return fail(RFA_E_INVALID, "out is null");
    *out = nullptr;
    if (!dims || !spacing_mm || !labels || !table) return fail(RFA_E_INVALID, "null argument");
    if (n_tissue < 1 || n_tissue > RFA_MAX_TISSUES) return fail(RFA_E_INVALID, "n_tissue %d outside 1..%d", n_tissue, RFA_MAX_TISSUES);
    if (batch < 1) return fail(RFA_E_INVALID, "batch must be >= 1");
    if (!(dt_s > 0.f) || !std::isfinite(dt_s)) return fail(RFA_E_INVALID, "dt must be positive and finite");
    if (!std::isfinite(t_blood_c)) return fail(RFA_E_INVALID, "t_blood must be finite");
    WsLayout L;
    if (!ws_layout(dims, batch, L)) return fail(RFA_E_INVALID, "dims must be positive (and the volume of sane size)");
    for (int a = 0; a < 3; ++a)
        if (!(spacing_mm[a] > 0.f) || !std::isfinite(spacing_mm[a])) return fail(RFA_E_INVALID, "spacing must be positive and finite");
    for (int l = 0; l < n_tissue; ++l)
        if (!tissue_ok(table[l])) return fail(RFA_E_INVALID, "tissue row %d: non-finite or non-positive constants", l);
    const size_t nvox = (size_t)dims[0] * dims[1] * dims[2];
    // Range check of the label ids on the host: a plain byte maximum over the volume (~4 ms for the 67 M voxels of C4).
    // It runs only when there is no device to do it: with a device the histogram kernel below finds an id >= n_tissue
    // after the upload (rfa_init_kernel masks the id to 4 bits, so a bad volume is never used as an index), and the
    // host walk would just delay the upload.
    auto host_label_check = [&]() -> int {
        unsigned char m[64] = {0};
        size_t v = 0;
        for (; v + 64 <= nvox; v += 64)
            for (int c = 0; c < 64; ++c) m[c] = labels[v + c] > m[c] ? labels[v + c] : m[c];
        unsigned mx = 0;
        for (; v < nvox; ++v) mx = labels[v] > mx ? labels[v] : mx;
        for (int c = 0; c < 64; ++c) mx = m[c] > mx ? m[c] : mx;
        if ((int)mx >= n_tissue) return fail(RFA_E_INVALID, "label id %u >= n_tissue %d", mx, n_tissue);
        return RFA_OK;
    };
    const double stab = rfa_stability_number(spacing_mm, table, n_tissue, dt_s);
    if (stab < 0) return fail(RFA_E_INVALID, "invalid constants");
    if (stab > 1.0)
        return fail(RFA_E_UNSTABLE, "dt = %g s violates the monotone bound: dt*(2 alpha sum 1/h^2 + beta/(rho cp)) = %.4f > 1", (double)dt_s, stab);
    if (workspace) {
        if (workspace_bytes < L.total) return fail(RFA_E_INVALID, "workspace of %zu bytes < required %zu", workspace_bytes, L.total);
        if (((uintptr_t)workspace & 255) != 0) return fail(RFA_E_INVALID, "workspace must be 256-byte aligned");
    }

    rfa_sim *s = new (std::nothrow) rfa_sim;
    if (!s) return fail(RFA_E_NOMEM, "host allocation failed");
    s->g.nx = dims[0];
    s->g.ny = dims[1];
    s->g.nz = dims[2];
    s->g.batch = batch;
    s->nvox = nvox;
    double W = 0;
    for (int a = 0; a < 3; ++a) {
        s->h_m[a] = (double)spacing_mm[a] * 1.0e-3;          // mm -> m (PAPER.md:115 vs :104)
        W += 1.0 / (s->h_m[a] * s->h_m[a]);
    }
    {
        // weights on the 2^-24 grid with an exact unit sum (rfa_device.cuh); the largest absorbs the residue
        const double q = 16777216.0;
        double w[3], wq[3];
        int big = 0;
        for (int a = 0; a < 3; ++a) {
            w[a] = 1.0 / (s->h_m[a] * s->h_m[a]) / W;
            wq[a] = std::nearbyint(w[a] * q) / q;
            if (w[a] > w[big]) big = a;
        }
        wq[big] = 1.0 - wq[(big + 1) % 3] - wq[(big + 2) % 3];
        s->g.wx = (float)wq[0];
        s->g.wy = (float)wq[1];
        s->g.wz = (float)wq[2];
    }
    s->dt = dt_s;
    s->t_blood = t_blood_c;
    s->g.t_blood = t_blood_c;
    s->g.thr = (float)(60.0 - (double)t_blood_c);            // T >= 60 C  (R-11)
    s->table.assign(table, table + n_tissue);
    for (int l = 0; l < n_tissue; ++l)
        if (table[l].flags & RFA_TISSUE_HELD) s->label_held_mask |= 1u << l;
    s->q_power.assign(batch, 0.0);
    s->stream = (cudaStream_t)cuda_stream;

    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev < 1) {
        delete s;
        cudaGetLastError();
        if (int lrc = host_label_check()) return lrc;       // invalid input is reported as such even without a device
        return fail(RFA_E_CUDA, "no CUDA device (%s); librfa has no CPU fallback", e != cudaSuccess ? cudaGetErrorString(e) : "count = 0");
    }
    if (cudaGetDevice(&s->device) != cudaSuccess) {
        delete s;
        cudaGetLastError();
        return fail(RFA_E_CUDA, "cudaGetDevice failed");
    }
    if (workspace) {
        cudaPointerAttributes at{};
        if (cudaPointerGetAttributes(&at, workspace) != cudaSuccess ||
            (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged)) {
            delete s;
            cudaGetLastError();
            return fail(RFA_E_INVALID, "workspace is not device memory");
        }
        if (at.type == cudaMemoryTypeDevice && at.device != s->device) {
            delete s;
            return fail(RFA_E_INVALID, "workspace lives on device %d, the current device is %d", at.device, s->device);
        }
        s->ws = (unsigned char *)workspace;
    } else {
        e = cudaMalloc((void **)&s->ws, L.total);
        if (e != cudaSuccess) {
            delete s;
            cudaGetLastError();
            return fail(RFA_E_NOMEM, "cudaMalloc of %zu bytes failed: %s", L.total, cudaGetErrorString(e));
        }
        s->own_ws = true;
    }
    s->theta[0] = (float *)(s->ws + L.theta0);
    s->theta[1] = (float *)(s->ws + L.theta1);
    s->resid[0] = s->ws + L.resid0;
    s->resid[1] = s->ws + L.resid1;
    s->state = s->ws + L.state;
    s->tables = (float *)(s->ws + L.tables);
    s->kap = (float *)(s->ws + L.kap);
    s->scratch = s->ws + L.scratch;
    s->counters = (unsigned long long *)(s->ws + L.counters);

    int rc = RFA_OK;
    do {
        // labels -> device (staged through scratch), then label -> initial temperature image
        e = cudaMemsetAsync(s->counters, 0, 256, s->stream);   // necrotic-voxel counts [0..1], dynamic work counter [4], hot warp-planes [5]
        if (e != cudaSuccess) { rc = cuda_fail(e, "counter reset"); break; }
        // feedback channel of the residual-prefetch choice; without it the variant simply stays off
        if (cudaHostAlloc((void **)&s->hot_host, 64, cudaHostAllocDefault) != cudaSuccess) { cudaGetLastError(); s->hot_host = nullptr; }
        else *s->hot_host = 0;
        if (cudaEventCreateWithFlags(&s->hot_evt, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); s->hot_evt = nullptr; }
        e = cudaMemcpyAsync(s->scratch, labels, nvox, cudaMemcpyHostToDevice, s->stream);
        if (e != cudaSuccess) { rc = cuda_fail(e, "label upload"); break; }
        float theta0[RFA_NLABEL], kl[RFA_NLABEL], kap[RFA_NLABEL * RFA_NLABEL];
        for (int l = 0; l < RFA_NLABEL; ++l) {
            theta0[l] = l < n_tissue ? (float)((double)table[l].t_init - (double)t_blood_c) : 0.f;
            kl[l] = l < n_tissue ? table[l].k : 0.f;
        }
        // face factors Kf/K_c - 1 = 2 K_n/(K_c + K_n) - 1 in fp64, rounded once; exactly 0 for equal K
        for (int c = 0; c < RFA_NLABEL; ++c)
            for (int n = 0; n < RFA_NLABEL; ++n) {
                double v = 0.0;
                if (c < n_tissue && n < n_tissue && table[c].k != table[n].k && (double)table[c].k + (double)table[n].k > 0.0)
                    v = 2.0 * (double)table[n].k / ((double)table[c].k + (double)table[n].k) - 1.0;
                kap[c * RFA_NLABEL + n] = (float)v;
            }
        e = cudaMemcpyAsync(s->kap, kap, sizeof kap, cudaMemcpyHostToDevice, s->stream);
        if (e != cudaSuccess) { rc = cuda_fail(e, "face table upload"); break; }
        // histogram of the label ids, on the device (held share below)
        unsigned long long *hist_dev = s->counters + 32;
        e = rfa_launch_label_hist(s->g, s->scratch, hist_dev, s->stream);
        s->launches++;
        if (e != cudaSuccess) { rc = cuda_fail(e, "label histogram"); break; }
        e = rfa_launch_init(s->g, s->scratch, theta0, kl, s->theta[0], s->resid[0], s->state, s->stream);
        s->launches++;
        if (e != cudaSuccess) { rc = cuda_fail(e, "init kernel"); break; }
        for (int b = 0; b < batch && rc == RFA_OK; ++b) rc = upload_table(s, b);
        if (rc != RFA_OK) break;
        make_plans(s);
        s->fused = default_fused(s);
        unsigned long long hist[256];
        e = cudaMemcpyAsync(hist, hist_dev, sizeof hist, cudaMemcpyDeviceToHost, s->stream);
        if (e != cudaSuccess) { rc = cuda_fail(e, "histogram download"); break; }
        e = cudaStreamSynchronize(s->stream);
        if (e != cudaSuccess) { rc = cuda_fail(e, "create"); break; }
        for (int l = 255; l >= n_tissue; --l)
            if (hist[l]) { rc = fail(RFA_E_INVALID, "label id %d >= n_tissue %d", l, n_tissue); break; }
        if (rc != RFA_OK) break;
        // Held-copy kernel variant (warps whose voxels are all held copy their rows instead of evaluating the
        // bracket; bit-identical): worth its extra vote per level only where a good part of the volume is held
        // (the air around the body in C4: +11 %; -7 % on the 128^3 phantoms without it).  rfa_configure_held_copy overrides.
        unsigned long long n_held = 0;
        for (int l = 0; l < n_tissue; ++l)
            if (table[l].flags & RFA_TISSUE_HELD) n_held += hist[l];
        s->held_copy_auto = n_held * 8 >= (unsigned long long)nvox ? 1 : 0;
        s->g.held_copy = s->held_copy_auto;
    } while (0);
    if (rc != RFA_OK) {
        const std::string msg = g_err;                     // keep the message of the failure, not of the clean-up
        cudaStreamSynchronize(s->stream);
        cudaGetLastError();
        if (s->hot_host) cudaFreeHost(s->hot_host);
        if (s->hot_evt) cudaEventDestroy(s->hot_evt);
        if (s->own_ws) cudaFree(s->ws);
        delete s;
        g_err = msg;
        return rc;
    }
    *out = s;
    return RFA_OK;
}

extern "C" void rfa_destroy(rfa_sim *s)
{
    if (!s) return;
    {
        DeviceGuard dg(s);
        cudaStreamSynchronize(s->stream);
        if (s->own_ws) cudaFree(s->ws);
        if (s->probes) cudaFree(s->probes);
        if (s->record) cudaFree(s->record);
        if (s->stage) cudaFree(s->stage);
        if (s->hot_host) cudaFreeHost(s->hot_host);
        if (s->hot_evt) cudaEventDestroy(s->hot_evt);
    }
    delete s;
}

extern "C" int rfa_set_needle(rfa_sim *s, int scenario, const float tip_mm[3], const float axis[3],
                              const uint8_t *mask, int mode, float value)
{
    int rc = check_sim(s, scenario);
    if (rc) return rc;
    DeviceGuard dg(s);
    if (mode != RFA_SRC_OFF && mode != RFA_SRC_DIRICHLET && mode != RFA_SRC_POWER) return fail(RFA_E_INVALID, "bad source mode %d", mode);
    if (mode != RFA_SRC_OFF && !mask) return fail(RFA_E_INVALID, "mask is null");
    if (mode != RFA_SRC_OFF && !std::isfinite(value)) return fail(RFA_E_INVALID, "source value must be finite");
    // tip / axis are metadata (the mask is authoritative), but a tip outside the grid or a non-unit axis means the
    // caller's geometry and its mask disagree: reject
    if (tip_mm) {
        const int n[3] = {s->g.nx, s->g.ny, s->g.nz};
        for (int a = 0; a < 3; ++a) {
            const double ext = n[a] * s->h_m[a] * 1.0e3;
            if (!std::isfinite(tip_mm[a]) || tip_mm[a] < -1.0e-3 || tip_mm[a] > ext + 1.0e-3)
                return fail(RFA_E_INVALID, "tip position %g mm outside the grid [0, %g] mm along axis %d", (double)tip_mm[a], ext, a);
        }
    }
    if (axis) {
        double n2 = 0;
        for (int a = 0; a < 3; ++a) {
            if (!std::isfinite(axis[a])) return fail(RFA_E_INVALID, "axis must be finite");
            n2 += (double)axis[a] * axis[a];
        }
        if (std::fabs(std::sqrt(n2) - 1.0) > 1.0e-3) return fail(RFA_E_INVALID, "axis must be a unit vector (|axis| = %.6f)", std::sqrt(n2));
    }
    const uint8_t *mdev = nullptr;
    cudaError_t e;
    if (mode != RFA_SRC_OFF) {
        if (is_device_ptr(mask)) {
            mdev = mask;
        } else {
            e = cudaMemcpyAsync(s->scratch, mask, s->nvox, cudaMemcpyHostToDevice, s->stream);
            if (e != cudaSuccess) return cuda_fail(e, "mask upload");
            mdev = s->scratch;
        }
    }
    const float theta_value = (float)((double)value - s->t_blood);
    e = rfa_launch_needle(s->g, scenario, mdev, mode, theta_value, s->theta[s->cur], s->resid[s->cur], s->state, s->stream);
    s->launches++;
    if (e != cudaSuccess) return cuda_fail(e, "needle kernel");
    s->q_power[scenario] = (mode == RFA_SRC_POWER) ? (double)value : 0.0;
    rc = upload_table(s, scenario);
    if (rc) return rc;
    if (mdev == s->scratch) {                               // the host mask may be reused by the caller
        e = cudaStreamSynchronize(s->stream);
        if (e != cudaSuccess) return cuda_fail(e, "set_needle");
    }
    return RFA_OK;
}

extern "C" int rfa_set_temperature(rfa_sim *s, int scenario, const float *t_c)
{
    int rc = check_sim(s, scenario);
    if (rc) return rc;
    DeviceGuard dg(s);
    if (!t_c) return fail(RFA_E_INVALID, "t_c is null");
    const float *src = t_c;
    cudaError_t e;
    const bool dev = is_device_ptr(t_c);
    if (!dev) {
        e = cudaMemcpyAsync(s->scratch, t_c, s->nvox * 4, cudaMemcpyHostToDevice, s->stream);
        if (e != cudaSuccess) return cuda_fail(e, "temperature upload");
        src = (const float *)s->scratch;
    }
    e = rfa_launch_set_temperature(s->g, scenario, src, s->theta[s->cur], s->resid[s->cur], s->state, s->stream);
    s->launches++;
    if (e != cudaSuccess) return cuda_fail(e, "set_temperature kernel");
    if (!dev) {
        e = cudaStreamSynchronize(s->stream);
        if (e != cudaSuccess) return cuda_fail(e, "set_temperature");
    }
    return RFA_OK;
}

// the TMA-staged one-step kernel serves single-step launches in Eq. 12 mode on grids with a TMA path
static bool can_stream(const rfa_sim *s) { return s->stream_ok && s->conduction == RFA_COND_EQ12; }

// what a launch of `did` time steps runs, given the configured kernel
static int kernel_for(const rfa_sim *s, int did)
{
    if (s->kernel == RFA_KERNEL_PLAIN) return RFA_KERNEL_PLAIN;
    if (did == 1 && can_stream(s) && (s->kernel == RFA_KERNEL_AUTO || s->kernel == RFA_KERNEL_STREAM)) return RFA_KERNEL_STREAM;
    if (s->kernel == RFA_KERNEL_STREAM) return s->plans()[1].ok ? RFA_KERNEL_BLOCKED : RFA_KERNEL_PLAIN;   // e.g. after rfa_set_conduction
    return s->plans()[did].ok ? RFA_KERNEL_BLOCKED : RFA_KERNEL_PLAIN;
}

extern "C" int rfa_configure(rfa_sim *s, int kernel, int fused_steps)
{
    if (!s) return fail(RFA_E_INVALID, "null simulation handle");
    if (kernel != RFA_KERNEL_AUTO && kernel != RFA_KERNEL_PLAIN && kernel != RFA_KERNEL_BLOCKED && kernel != RFA_KERNEL_STREAM)
        return fail(RFA_E_INVALID, "bad kernel id %d", kernel);
    if (fused_steps < 0 || fused_steps > 4) return fail(RFA_E_INVALID, "fused_steps must be 0..4");
    int f = fused_steps == 0 ? default_fused(s) : fused_steps;
    if (kernel == RFA_KERNEL_STREAM) {
        if (!can_stream(s))
            return fail(RFA_E_INVALID, "the TMA-staged one-step kernel needs nx %% 16 == 0 and the Eq. 12 conduction term (grid %dx%dx%d)", s->g.nx, s->g.ny, s->g.nz);
        if (fused_steps > 1) return fail(RFA_E_INVALID, "the one-step kernel takes fused_steps 0 or 1");
        f = 1;
    }
    if (kernel == RFA_KERNEL_BLOCKED && !s->plans()[f].ok)
        return fail(RFA_E_INVALID, "the blocked kernel needs nx %% 4 == 0 and ny, nz >= fused steps (grid %dx%dx%d, fused %d)", s->g.nx, s->g.ny, s->g.nz, f);
    s->kernel = kernel;
    s->fused = f;
    return RFA_OK;
}

extern "C" int rfa_configure_held_copy(rfa_sim *s, int mode)
{
    if (!s) return fail(RFA_E_INVALID, "null simulation handle");
    if (mode != RFA_HELD_COPY_AUTO && mode != RFA_HELD_COPY_OFF && mode != RFA_HELD_COPY_ON)
        return fail(RFA_E_INVALID, "bad held-copy mode %d", mode);
    s->g.held_copy = mode == RFA_HELD_COPY_AUTO ? s->held_copy_auto : (mode == RFA_HELD_COPY_ON ? 1 : 0);
    return RFA_OK;
}

extern "C" int rfa_configure_staging(rfa_sim *s, int mode)
{
    if (!s) return fail(RFA_E_INVALID, "null simulation handle");
    if (mode != RFA_STAGING_AUTO && mode != RFA_STAGING_CP_ASYNC && mode != RFA_STAGING_TMA)
        return fail(RFA_E_INVALID, "bad staging mode %d", mode);
    DeviceGuard dg(s);
    const int old = s->staging;
    s->staging = mode;
    make_plans(s);
    if (mode == RFA_STAGING_TMA && !(s->plans_by_mode[0][2].tma || s->plans_by_mode[0][3].tma)) {
        s->staging = old;
        make_plans(s);
        return fail(RFA_E_INVALID, "no TMA-staged variant for this grid (needs nx %% 16 == 0, ny even; grid %dx%dx%d)", s->g.nx, s->g.ny, s->g.nz);
    }
    if (s->kernel == RFA_KERNEL_BLOCKED && !s->plans()[s->fused].ok) s->kernel = RFA_KERNEL_AUTO;
    return RFA_OK;
}

extern "C" int rfa_configure_residual_prefetch(rfa_sim *s, int mode)
{
    if (!s) return fail(RFA_E_INVALID, "null simulation handle");
    if (mode != RFA_RES_PREFETCH_AUTO && mode != RFA_RES_PREFETCH_OFF && mode != RFA_RES_PREFETCH_ON)
        return fail(RFA_E_INVALID, "bad residual-prefetch mode %d", mode);
    s->res_prefetch_mode = mode;
    return RFA_OK;
}

extern "C" int rfa_query_hot_fraction(rfa_sim *s, double *fraction, int *prefetch_on)
{
    if (!s) return fail(RFA_E_INVALID, "null simulation handle");
    if (fraction) *fraction = s->hot_fraction;
    if (prefetch_on) *prefetch_on = s->res_prefetch_mode == RFA_RES_PREFETCH_AUTO ? s->res_prefetch_on : s->res_prefetch_mode;
    return RFA_OK;
}

extern "C" int rfa_configure_tile(rfa_sim *s, int shape)
{
    if (!s) return fail(RFA_E_INVALID, "null simulation handle");
    if (shape < -1 || shape >= RFA_N_SHAPES) return fail(RFA_E_INVALID, "tile shape must be -1 (planner's choice), 0 (64 x 32) or 1 (128 x 16)");
    DeviceGuard dg(s);
    const int old = s->force_shape;
    s->force_shape = shape;
    make_plans(s);
    // a forced shape that cannot run is refused whatever the kernel setting: under RFA_KERNEL_AUTO it would otherwise
    // drop to the plain kernel without a word (only RFA_KERNEL_PLAIN, which has no tiles, takes any shape)
    if (shape != -1 && s->kernel != RFA_KERNEL_PLAIN && !s->plans()[s->fused].ok) {
        s->force_shape = old;
        make_plans(s);
        return fail(RFA_E_INVALID, "tile shape %d cannot run the configured %d fused steps on this grid", shape, s->fused);
    }
    return RFA_OK;
}

extern "C" int rfa_set_conduction(rfa_sim *s, int mode)
{
    if (!s) return fail(RFA_E_INVALID, "null simulation handle");
    if (mode != RFA_COND_EQ12 && mode != RFA_COND_FACE) return fail(RFA_E_INVALID, "bad conduction mode %d", mode);
    if (mode == RFA_COND_FACE) {
        // monotone bound with the largest face conductivity a voxel of each label can see (R-18, R-28)
        double W = 0, kmax = 0, worst = 0;
        for (int a = 0; a < 3; ++a) W += 1.0 / (s->h_m[a] * s->h_m[a]);
        for (const rfa_tissue &t : s->table) kmax = std::max(kmax, (double)t.k);
        for (const rfa_tissue &t : s->table) {
            if (t.flags & RFA_TISSUE_HELD) continue;
            const double rc = (double)t.rho * t.cp, kf = 2.0 * (double)t.k * kmax / ((double)t.k + kmax);
            worst = std::max(worst, s->dt * (2.0 * kf / rc * W + (double)t.wb_cb / rc));
        }
        if (worst > 1.0)
            return fail(RFA_E_UNSTABLE, "dt = %g s violates the monotone bound with face conductivities: %.4f > 1", s->dt, worst);
    }
    s->conduction = mode;
    return RFA_OK;
}

extern "C" int rfa_query(rfa_sim *s, int *kernel, int *fused_steps, int64_t *kernel_launches)
{
    if (!s) return fail(RFA_E_INVALID, "null simulation handle");
    const int k = kernel_for(s, s->fused);
    if (kernel) *kernel = k;
    if (fused_steps) *fused_steps = k == RFA_KERNEL_BLOCKED ? s->fused : 1;
    if (kernel_launches) *kernel_launches = s->launches;
    return RFA_OK;
}

// Feedback for the residual-prefetch variant: every RFA_HOT_SAMPLE_EVERY launches the hot warp-plane counter is copied to
// pinned memory behind the launches issued so far; a later call finds the copy complete (cudaEventQuery, never a wait) and
// switches the variant on above RFA_HOT_ON of the warp-planes, off below RFA_HOT_OFF.  Both variants give bit-identical
// fields, so the switch changes speed only.  Measured on the B200: the variant costs 2.4 % where next to nothing is hot
// (C4: 0.17 % of the warp-planes, 770 -> 752 GVox/s), is neutral at 1.1 % (C5), gains 8 % at 2.2 % (C3 after 3000
// steps, 452 -> 487) and 11 % at 84 % (C4F, 290 -> 322): break-even near 0.5 %.
#define RFA_HOT_SAMPLE_EVERY 32
#define RFA_HOT_ON 0.004
#define RFA_HOT_OFF 0.0025
static void sample_hot_fraction(rfa_sim *s, const RfaTbPlan &pl)
{
    s->planes_issued += (double)pl.n_items * (pl.zchunk + 2 * pl.fused) * 8.0;       // 8 warps per CTA
    if (!s->hot_host || !s->hot_evt) return;
    if (s->hot_pending) {
        ++s->launches_since_sample;
        if (s->res_prefetch_mode == RFA_RES_PREFETCH_AUTO && s->launches_since_sample >= 2 * RFA_HOT_SAMPLE_EVERY) {
            // The host has run RFA_HOT_SAMPLE_EVERY launches past the sample and the device has not reached it yet: wait for
            // it here.  The device still has those launches queued, so it never idles; the host just stops running further
            // ahead of it than the feedback can follow (a single rfa_step(12000) would otherwise issue every launch with
            // the choice made before the first one ran).
            if (cudaEventSynchronize(s->hot_evt) != cudaSuccess) { cudaGetLastError(); return; }
        } else if (cudaEventQuery(s->hot_evt) != cudaSuccess) {
            cudaGetLastError();                              // not ready yet: ask again at the next launch
            return;
        }
        const unsigned long long now = *s->hot_host;
        const double planes = s->planes_at_sample - s->planes_seen;
        if (planes > 0) {
            s->hot_fraction = (double)(now - s->hot_seen) / planes;
            if (s->hot_fraction >= RFA_HOT_ON) s->res_prefetch_on = 1;
            else if (s->hot_fraction < RFA_HOT_OFF) s->res_prefetch_on = 0;
        }
        s->hot_seen = now;
        s->planes_seen = s->planes_at_sample;
        s->hot_pending = false;
        s->launches_since_sample = 0;
        return;
    }
    if (++s->launches_since_sample >= RFA_HOT_SAMPLE_EVERY) {
        if (cudaMemcpyAsync(s->hot_host, s->counters + 5, sizeof(unsigned long long), cudaMemcpyDeviceToHost, s->stream) == cudaSuccess &&
            cudaEventRecord(s->hot_evt, s->stream) == cudaSuccess) {
            s->hot_pending = true;
            s->launches_since_sample = RFA_HOT_SAMPLE_EVERY;
            s->planes_at_sample = s->planes_issued;
        } else {
            cudaGetLastError();
        }
    }
}

// n time steps on the stream: launches of up to `fused` steps each, buffers swapped per launch (Alg. 2)
static int advance(rfa_sim *s, int n)
{
    const float *kap = s->conduction == RFA_COND_FACE ? s->kap : nullptr;
    const int fused = (s->kernel == RFA_KERNEL_PLAIN || s->kernel == RFA_KERNEL_STREAM) ? 1 : s->fused;
    while (n > 0) {
        cudaError_t e;
        int did = std::min(n, fused);
        while (did > 1 && !s->plans()[did].ok) --did;
        const int k = kernel_for(s, did);
        float *tin = s->theta[s->cur], *tout = s->theta[s->cur ^ 1];
        unsigned char *rin = s->resid[s->cur], *rout = s->resid[s->cur ^ 1];
        if (k == RFA_KERNEL_STREAM)
        {
            e = rfa_launch_stream(s->g, s->stream_plan, s->tm_theta[s->cur], s->tm_state, tout, rin, rout, s->state, s->tables,
                                  s->counters + 4, s->stream_draws, s->stream);
            // every launch that ran draws exactly n_items times; one that was never queued drew nothing, and counting it
            // would hand every later launch a work_base ahead of the device counter (items skipped or done twice)
            if (e == cudaSuccess) s->stream_draws += (unsigned long long)s->stream_plan.n_items;
        }
        else if (k == RFA_KERNEL_BLOCKED) {
            const RfaTbPlan &pl = s->plans()[did];
            const int rpf = s->res_prefetch_mode == RFA_RES_PREFETCH_AUTO ? s->res_prefetch_on : s->res_prefetch_mode;
            e = rfa_launch_blocked(s->g, pl, tin, tout, rin, rout, s->state, s->tables, kap, &s->tm_blk_theta[s->cur][pl.shape],
                                   &s->tm_blk_state[pl.shape], rpf && rfa_blocked_has_prefetch(did, pl.tma), s->counters + 5, s->stream);
            if (e == cudaSuccess) sample_hot_fraction(s, pl);
        }
        else {
            did = 1;
            e = rfa_launch_plain(s->g, tin, tout, rin, rout, s->state, s->tables, kap, s->stream);
        }
        s->launches++;
        if (e != cudaSuccess) return cuda_fail(e, "step kernel");
        s->cur ^= 1;                                        // Alg. 2: swap the two buffers
        n -= did;
    }
    return RFA_OK;
}

extern "C" int rfa_query_variant(rfa_sim *s, int out[8])
{
    if (!s || !out) return fail(RFA_E_INVALID, "null argument");
    const int k = kernel_for(s, s->fused);
    const RfaTbPlan &p = s->plans()[s->fused];
    const bool blocked = k == RFA_KERNEL_BLOCKED, stream = k == RFA_KERNEL_STREAM;
    out[0] = blocked ? s->fused : 1;
    out[1] = blocked ? 4 * RFA_TB_SHAPE[p.shape][s->fused].tx : (stream ? RFA_STREAM_BX : 0);
    out[2] = blocked ? RFA_TB_SHAPE[p.shape][s->fused].ry * RFA_TB_SHAPE[p.shape][s->fused].ty : (stream ? RFA_STREAM_BY : 0);
    out[3] = blocked ? p.grid : (stream ? s->stream_plan.grid : 0);
    out[4] = (blocked || stream) ? s->g.held_copy : 0;
    out[5] = s->conduction;
    out[6] = stream ? RFA_STAGING_TMA : (blocked && p.tma ? RFA_STAGING_TMA : RFA_STAGING_CP_ASYNC);
    const int rpf = s->res_prefetch_mode == RFA_RES_PREFETCH_AUTO ? s->res_prefetch_on : s->res_prefetch_mode;
    out[7] = (blocked && rpf && rfa_blocked_has_prefetch(s->fused, p.tma)) ? 1 : 0;
    return RFA_OK;
}

extern "C" int rfa_step(rfa_sim *s, int n)
{
    if (!s) return fail(RFA_E_INVALID, "null simulation handle");
    DeviceGuard dg(s);
    if (n < 0) return fail(RFA_E_INVALID, "n must be >= 0");
    return advance(s, n);
}

extern "C" int rfa_set_probes(rfa_sim *s, int n_probes, const int64_t *index)
{
    if (!s) return fail(RFA_E_INVALID, "null simulation handle");
    DeviceGuard dg(s);
    if (n_probes < 0 || (n_probes > 0 && !index)) return fail(RFA_E_INVALID, "bad probe list");
    const long long total = (long long)s->nvox * s->g.batch;
    for (int p = 0; p < n_probes; ++p)
        if (index[p] < 0 || index[p] >= total) return fail(RFA_E_INVALID, "probe %d: index %lld outside [0,%lld)", p, (long long)index[p], total);
    cudaError_t e = cudaStreamSynchronize(s->stream);       // an earlier record may still read the old list
    if (e != cudaSuccess) return cuda_fail(e, "set_probes");
    if (s->probes) cudaFree(s->probes);
    s->probes = nullptr;
    s->n_probes = 0;
    if (n_probes == 0) return RFA_OK;
    e = cudaMalloc((void **)&s->probes, (size_t)n_probes * sizeof(long long));
    if (e != cudaSuccess) { cudaGetLastError(); return fail(RFA_E_NOMEM, "cudaMalloc of the probe list failed"); }
    static_assert(sizeof(long long) == sizeof(int64_t), "probe indices are 64-bit");
    e = cudaMemcpy(s->probes, index, (size_t)n_probes * sizeof(long long), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return cuda_fail(e, "probe upload");
    s->n_probes = n_probes;
    return RFA_OK;
}

extern "C" int rfa_step_record(rfa_sim *s, int n, int every, float *out)
{
    if (!s) return fail(RFA_E_INVALID, "null simulation handle");
    DeviceGuard dg(s);
    if (n < 0 || every < 1 || (n % every) != 0) return fail(RFA_E_INVALID, "n must be a non-negative multiple of every >= 1");
    if (s->n_probes == 0) return fail(RFA_E_INVALID, "no probes set (rfa_set_probes)");
    if (!out) return fail(RFA_E_INVALID, "out is null");
    const size_t rows = (size_t)(n / every), need = rows * (size_t)s->n_probes;
    if (rows == 0) return RFA_OK;
    const bool dev = is_device_ptr(out);
    float *dst = out;
    cudaError_t e;
    if (!dev) {
        if (s->record_cap < need) {
            e = cudaStreamSynchronize(s->stream);
            if (e != cudaSuccess) return cuda_fail(e, "step_record");
            if (s->record) cudaFree(s->record);
            s->record = nullptr;
            s->record_cap = 0;
            e = cudaMalloc((void **)&s->record, need * sizeof(float));
            if (e != cudaSuccess) { cudaGetLastError(); return fail(RFA_E_NOMEM, "cudaMalloc of %zu record floats failed", need); }
            s->record_cap = need;
        }
        dst = s->record;
    }
    for (size_t m = 0; m < rows; ++m) {
        int rc = advance(s, every);
        if (rc) return rc;
        e = rfa_launch_probe(s->g, s->n_probes, s->probes, s->theta[s->cur], dst + m * s->n_probes, s->stream);
        s->launches++;
        if (e != cudaSuccess) return cuda_fail(e, "probe kernel");
    }
    if (!dev) {
        e = cudaMemcpyAsync(out, dst, need * sizeof(float), cudaMemcpyDeviceToHost, s->stream);
        if (e != cudaSuccess) return cuda_fail(e, "record download");
    }
    e = cudaStreamSynchronize(s->stream);
    if (e != cudaSuccess) return cuda_fail(e, "step_record");
    return RFA_OK;
}

// rfa_step_record without any allocation: probe list and rows in the per-GPU static array of rfa_noalloc.cu (include/rfa.h
// says for whom).  No cudaMalloc / cudaFree / cudaMallocHost here or below: advance() only launches, the three
// rfa_static_record_* helpers only copy and launch.
extern "C" int rfa_step_record_static(rfa_sim *s, int n, int every, int n_probes, const int64_t *index, float *out)
{
    if (!s) return fail(RFA_E_INVALID, "null simulation handle");
    DeviceGuard dg(s);
    if (n < 0 || every < 1 || (n % every) != 0) return fail(RFA_E_INVALID, "n must be a non-negative multiple of every >= 1");
    if (n_probes < 1 || !index) return fail(RFA_E_INVALID, "need at least one probe and its index list");
    if (!out) return fail(RFA_E_INVALID, "out is null");
    if (n_probes > RFA_STATIC_RECORD_MAX_PROBES)
        return fail(RFA_E_INVALID, "%d probes: the static scratch holds at most %d (RFA_STATIC_RECORD_MAX_PROBES); use rfa_set_probes + rfa_step_record",
                    n_probes, (int)RFA_STATIC_RECORD_MAX_PROBES);
    const size_t rows = (size_t)(n / every), need = rows * (size_t)n_probes;
    if (need > (size_t)RFA_STATIC_RECORD_MAX_FLOATS)
        return fail(RFA_E_INVALID, "%zu records x %d probes = %zu floats: the static scratch holds at most %d (RFA_STATIC_RECORD_MAX_FLOATS); "
                    "record the run as several shorter calls", rows, n_probes, need, (int)RFA_STATIC_RECORD_MAX_FLOATS);
    const long long total = (long long)s->nvox * s->g.batch;
    for (int p = 0; p < n_probes; ++p)
        if (index[p] < 0 || index[p] >= total) return fail(RFA_E_INVALID, "probe %d: index %lld outside [0,%lld)", p, (long long)index[p], total);
    if (rows == 0) return RFA_OK;
    static_assert(sizeof(long long) == sizeof(int64_t), "probe indices are 64-bit");
    cudaError_t e = rfa_static_record_begin(n_probes, (const long long *)index, s->stream);
    if (e != cudaSuccess) return cuda_fail(e, "static scratch set-up / probe upload");
    for (size_t m = 0; m < rows; ++m) {
        int rc = advance(s, every);
        if (rc) return rc;
        e = rfa_static_record_probe(s->g, n_probes, s->theta[s->cur], m, s->stream);
        s->launches++;
        if (e != cudaSuccess) return cuda_fail(e, "probe kernel (static scratch)");
    }
    e = rfa_static_record_fetch(out, need, s->stream);
    if (e != cudaSuccess) return cuda_fail(e, "record download (static scratch)");
    e = cudaStreamSynchronize(s->stream);
    if (e != cudaSuccess) return cuda_fail(e, "step_record_static");
    return RFA_OK;
}

extern "C" int rfa_current_frame(rfa_sim *s, int scenario, const float **theta_dev, float *t_blood_c)
{
    int rc = check_sim(s, scenario);
    if (rc) return rc;
    DeviceGuard dg(s);
    if (!theta_dev) return fail(RFA_E_INVALID, "theta_dev is null");
    *theta_dev = s->theta[s->cur] + (size_t)scenario * s->nvox;
    if (t_blood_c) *t_blood_c = (float)s->t_blood;
    return RFA_OK;
}

extern "C" int rfa_warp_temperature(rfa_sim *s, int scenario, const float *disp, float scale, float *out)
{
    int rc = check_sim(s, scenario);
    if (rc) return rc;
    DeviceGuard dg(s);
    if (!disp || !out) return fail(RFA_E_INVALID, "null argument");
    if (!std::isfinite(scale)) return fail(RFA_E_INVALID, "scale must be finite");
    const size_t nvox = s->nvox;
    const float *ddev = disp;
    cudaError_t e;
    const bool din = is_device_ptr(disp), dev = is_device_ptr(out);
    if (!din) {
        // host field: staged through the library-owned buffer (kept for the next call, freed by rfa_destroy)
        rc = ensure_stage(s, 3 * nvox);
        if (rc) return fail(rc, "staging buffer for the displacement field (%zu floats)", 3 * nvox);
        e = cudaMemcpyAsync(s->stage, disp, 3 * nvox * sizeof(float), cudaMemcpyHostToDevice, s->stream);
        if (e != cudaSuccess) return cuda_fail(e, "displacement upload");
        ddev = s->stage;
    }
    float *dst = dev ? out : (float *)s->scratch;
    const float inv_h[3] = {(float)(1.0e-3 / s->h_m[0]), (float)(1.0e-3 / s->h_m[1]), (float)(1.0e-3 / s->h_m[2])};
    e = rfa_launch_warp(s->g, scenario, s->theta[s->cur], ddev, scale, inv_h, dst, s->stream);
    s->launches++;
    if (e != cudaSuccess) return cuda_fail(e, "warp kernel");
    if (!dev) {
        e = cudaMemcpyAsync(out, dst, nvox * sizeof(float), cudaMemcpyDeviceToHost, s->stream);
        if (e != cudaSuccess) return cuda_fail(e, "warp download");
    }
    // device field in, device image out: nothing of the caller's host memory is touched -> asynchronous
    if (!din || !dev) {
        e = cudaStreamSynchronize(s->stream);
        if (e != cudaSuccess) return cuda_fail(e, "warp_temperature");
    }
    return RFA_OK;
}

extern "C" int rfa_render_zone(rfa_sim *s, int scenario, const rfa_view *view, float *tmax, float *depth)
{
    int rc = check_sim(s, scenario);
    if (rc) return rc;
    DeviceGuard dg(s);
    if (!view || !tmax) return fail(RFA_E_INVALID, "null argument");
    if (view->width < 1 || view->height < 1 || (long long)view->width * view->height > (1LL << 28))
        return fail(RFA_E_INVALID, "image of %d x %d pixels: need 1 <= W*H <= 2^28", view->width, view->height);
    if (!(view->pixel_mm > 0.f) || !(view->step_mm > 0.f) || !std::isfinite(view->pixel_mm) || !std::isfinite(view->step_mm) ||
        !std::isfinite(view->iso_c))
        return fail(RFA_E_INVALID, "pixel_mm and step_mm must be positive and finite, iso_c finite");
    RfaRay ray{};
    double w[3], up[3], n2 = 0;
    for (int a = 0; a < 3; ++a) {
        if (!std::isfinite(view->dir[a]) || !std::isfinite(view->up[a])) return fail(RFA_E_INVALID, "dir / up must be finite");
        w[a] = view->dir[a];
        up[a] = view->up[a];
        n2 += w[a] * w[a];
    }
    if (!(n2 > 0)) return fail(RFA_E_INVALID, "dir must not be zero");
    for (int a = 0; a < 3; ++a) w[a] /= std::sqrt(n2);
    double e1[3] = {up[1] * w[2] - up[2] * w[1], up[2] * w[0] - up[0] * w[2], up[0] * w[1] - up[1] * w[0]};   // up x dir
    const double l1 = std::sqrt(e1[0] * e1[0] + e1[1] * e1[1] + e1[2] * e1[2]);
    if (!(l1 > 1e-12)) return fail(RFA_E_INVALID, "up must not be parallel to dir");
    for (int a = 0; a < 3; ++a) e1[a] /= l1;
    const double e2[3] = {w[1] * e1[2] - w[2] * e1[1], w[2] * e1[0] - w[0] * e1[2], w[0] * e1[1] - w[1] * e1[0]};   // dir x e1
    const int n[3] = {s->g.nx, s->g.ny, s->g.nz};
    double diag2 = 0;
    for (int a = 0; a < 3; ++a) {
        const double h_mm = s->h_m[a] * 1.0e3;
        ray.c[a] = 0.5 * n[a] * h_mm;
        ray.e1[a] = e1[a];
        ray.e2[a] = e2[a];
        ray.w[a] = w[a];
        ray.inv_h[a] = 1.0 / h_mm;
        diag2 += (n[a] * h_mm) * (n[a] * h_mm);
    }
    ray.R = 0.5 * std::sqrt(diag2);
    ray.pixel = view->pixel_mm;
    ray.step = view->step_mm;
    ray.width = view->width;
    ray.height = view->height;
    const double ns = std::floor(2.0 * ray.R / ray.step) + 1.0;
    if (ns > 1.0e6) return fail(RFA_E_INVALID, "step_mm too small: %.0f samples per ray", ns);
    ray.n_samples = (int)ns;
    const size_t npix = (size_t)view->width * view->height;
    // host outputs are staged in the library-owned staging buffer (grows on demand): tmax first, depth behind it
    const bool tdev = is_device_ptr(tmax), ddev = depth ? is_device_ptr(depth) : true;
    const size_t n_staged = (tdev ? 0 : npix) + ((depth && !ddev) ? npix : 0);
    if (n_staged) {
        rc = ensure_stage(s, n_staged);
        if (rc) return fail(rc, "staging buffer for the images (%zu floats)", n_staged);
    }
    float *tdst = tdev ? tmax : s->stage;
    float *ddst = depth ? (ddev ? depth : s->stage + (tdev ? 0 : npix)) : nullptr;
    const float iso_theta = (float)((double)view->iso_c - s->t_blood);
    cudaError_t e = rfa_launch_render(s->g, scenario, ray, s->theta[s->cur], iso_theta, tdst, ddst, s->stream);
    s->launches++;
    if (e != cudaSuccess) return cuda_fail(e, "render kernel");
    if (!tdev) e = cudaMemcpyAsync(tmax, tdst, npix * sizeof(float), cudaMemcpyDeviceToHost, s->stream);
    if (e == cudaSuccess && depth && !ddev) e = cudaMemcpyAsync(depth, ddst, npix * sizeof(float), cudaMemcpyDeviceToHost, s->stream);
    if (e != cudaSuccess) return cuda_fail(e, "render download");
    e = cudaStreamSynchronize(s->stream);
    if (e != cudaSuccess) return cuda_fail(e, "render_zone");
    return RFA_OK;
}

extern "C" int rfa_synchronize(rfa_sim *s)
{
    if (!s) return fail(RFA_E_INVALID, "null simulation handle");
    DeviceGuard dg(s);
    cudaError_t e = cudaStreamSynchronize(s->stream);
    if (e != cudaSuccess) return cuda_fail(e, "synchronize");
    return RFA_OK;
}

extern "C" int rfa_get_temperature(rfa_sim *s, int scenario, float *out)
{
    int rc = check_sim(s, scenario);
    if (rc) return rc;
    DeviceGuard dg(s);
    if (!out) return fail(RFA_E_INVALID, "out is null");
    const bool dev = is_device_ptr(out);
    float *dst = dev ? out : (float *)s->scratch;
    cudaError_t e = rfa_launch_get_temperature(s->g, scenario, s->theta[s->cur], dst, s->stream);
    s->launches++;
    if (e != cudaSuccess) return cuda_fail(e, "get_temperature kernel");
    if (!dev) {
        e = cudaMemcpyAsync(out, dst, s->nvox * 4, cudaMemcpyDeviceToHost, s->stream);
        if (e != cudaSuccess) return cuda_fail(e, "temperature download");
    }
    e = cudaStreamSynchronize(s->stream);
    if (e != cudaSuccess) return cuda_fail(e, "get_temperature");
    return RFA_OK;
}

extern "C" int rfa_get_necrosis(rfa_sim *s, int scenario, uint8_t *out)
{
    int rc = check_sim(s, scenario);
    if (rc) return rc;
    DeviceGuard dg(s);
    if (!out) return fail(RFA_E_INVALID, "out is null");
    const bool dev = is_device_ptr(out);
    uint8_t *dst = dev ? out : s->scratch;
    cudaError_t e = rfa_launch_get_necrosis(s->g, scenario, s->state, dst, s->stream);
    s->launches++;
    if (e != cudaSuccess) return cuda_fail(e, "get_necrosis kernel");
    if (!dev) {
        e = cudaMemcpyAsync(out, dst, s->nvox, cudaMemcpyDeviceToHost, s->stream);
        if (e != cudaSuccess) return cuda_fail(e, "necrosis download");
    }
    e = cudaStreamSynchronize(s->stream);
    if (e != cudaSuccess) return cuda_fail(e, "get_necrosis");
    return RFA_OK;
}

extern "C" int rfa_necrotic_voxels(rfa_sim *s, int scenario, int64_t *all_voxels, int64_t *tissue_voxels)
{
    int rc = check_sim(s, scenario);
    if (rc) return rc;
    DeviceGuard dg(s);
    cudaError_t e = rfa_launch_count(s->g, scenario, s->state, s->label_held_mask, s->counters, s->stream);
    s->launches++;
    if (e != cudaSuccess) return cuda_fail(e, "count kernel");
    unsigned long long h[2] = {0, 0};
    e = cudaMemcpyAsync(h, s->counters, sizeof h, cudaMemcpyDeviceToHost, s->stream);
    if (e != cudaSuccess) return cuda_fail(e, "count download");
    e = cudaStreamSynchronize(s->stream);
    if (e != cudaSuccess) return cuda_fail(e, "necrotic_voxels");
    if (all_voxels) *all_voxels = (int64_t)h[0];
    if (tissue_voxels) *tissue_voxels = (int64_t)h[1];
    return RFA_OK;
}
