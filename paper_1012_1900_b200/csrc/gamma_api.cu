// gamma_api.cu -- host side of libgamma_b200.so: argument checks, workspace, kernel launches.
// The C-ABI is documented in include/gamma_b200.h.  There is no CPU path here: every step of the hot path
// runs in the kernels of gamma_search.cuh / radix_sort.cuh / offset_table.cuh / stats.cuh.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <tuple>
#include <utility>

#include "../../include/gamma_b200.h"
#include "common.cuh"
#include "gamma_search.cuh"
#include "offset_table.cuh"
#include "radix_sort.cuh"
#include "stats.cuh"
#include "tile_star.cuh"
#include "general.cuh"

using namespace gamma_b200;

namespace {

thread_local std::string g_err;
std::mutex g_mu;

// Host-side time of the submission path (build with -DGAMMA_HOSTPROF; printed to stderr by gamma_release()).
#ifdef GAMMA_HOSTPROF
}  // namespace
#include <chrono>
namespace {
struct HostProf {
    double us[10] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    long long n[10] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
} g_hp;
const char* const HP_NAMES[10] = {"gamma_eval_ex total", "back-pressure wait", "kernel launches", "events", "prepare/order/ctl",
                                  "argument checks", "getenv", "enqueue_kernels", "graph node update", "graph launch"};
struct HpScope {
    int k;
    std::chrono::steady_clock::time_point t0;
    explicit HpScope(int k_) : k(k_), t0(std::chrono::steady_clock::now()) {}
    ~HpScope()
    {
        g_hp.us[k] += std::chrono::duration<double, std::micro>(std::chrono::steady_clock::now() - t0).count();
        ++g_hp.n[k];
    }
};
#define HP(k) HpScope hp_scope_##k(k)
#else
#define HP(k) do { } while (0)
#endif

int fail(int code, const std::string& msg)
{
    g_err = msg;
    return code;
}
#define CU_TRY(call)                                                                          \
    do {                                                                                      \
        cudaError_t e_ = (call);                                                              \
        if (e_ != cudaSuccess)                                                                \
            return fail(e_ == cudaErrorMemoryAllocation ? GAMMA_ERR_OUT_OF_MEMORY : GAMMA_ERR_CUDA, \
                        std::string(#call) + ": " + cudaGetErrorString(e_));                 \
    } while (0)


// A call's kernels as an instantiated CUDA graph whose kernel-node parameters are rewritten for every call
// (cudaGraphExecKernelNodeSetParams: 0.4 us per node, one graph launch of 1.3 us -- against 3.3 us per stream launch,
// measured on the B200 box): the host cost of a call on a lane stream.  While `g_upd` is set, launch_ex() does not
// launch: it checks that the kernel is the one the node was built from and stores the new grid and arguments.
// While `g_rec` is set (the capture that builds such a graph) it notes the kernels in launch order.
constexpr int UPD_MAX_NODES = 8;
struct GraphUpdate {
    cudaGraphExec_t exec;
    const cudaGraphNode_t* nodes;
    void* const* funcs;
    int count, idx;
    bool ok;
};
GraphUpdate* g_upd = nullptr;
struct LaunchRecord { void* funcs[UPD_MAX_NODES]; int count; bool overflow; };
LaunchRecord* g_rec = nullptr;

template <typename Tuple, size_t... I>
void tuple_pointers(Tuple& t, void** p, std::index_sequence<I...>)
{
    ((p[I] = const_cast<void*>(static_cast<const void*>(&std::get<I>(t)))), ...);
}

// Kernel launch with attributes: `pdl` = programmatic dependent launch (the kernel may start while its predecessor
// in the stream drains; it calls pdl_wait() before touching the predecessor's results), `coop` = cooperative
// (all blocks co-resident: required by the grid barrier of k_norm).
template <typename... KArgs, typename... Args>
cudaError_t launch_ex(void (*kernel)(KArgs...), int grid, int block, size_t smem, cudaStream_t st, bool pdl, bool coop,
                      Args... args)
{
    if (g_upd) {
        GraphUpdate& u = *g_upd;
        if (u.idx >= u.count || u.funcs[u.idx] != reinterpret_cast<void*>(kernel)) { u.ok = false; return cudaSuccess; }
        std::tuple<std::remove_cv_t<KArgs>...> vals(static_cast<KArgs>(args)...);
        void* ptrs[sizeof...(KArgs)];
        tuple_pointers(vals, ptrs, std::index_sequence_for<KArgs...>{});
        cudaKernelNodeParams kp = {};
        kp.func = reinterpret_cast<void*>(kernel);
        kp.gridDim = dim3((unsigned)grid); kp.blockDim = dim3((unsigned)block);
        kp.sharedMemBytes = (unsigned)smem; kp.kernelParams = ptrs; kp.extra = nullptr;
        HP(8);
        return cudaGraphExecKernelNodeSetParams(u.exec, u.nodes[u.idx++], &kp);
    }
    if (g_rec) {
        if (g_rec->count < UPD_MAX_NODES) g_rec->funcs[g_rec->count++] = reinterpret_cast<void*>(kernel);
        else g_rec->overflow = true;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)block);
    cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[2];
    unsigned n = 0;
    if (pdl) { at[n].id = cudaLaunchAttributeProgrammaticStreamSerialization; at[n].val.programmaticStreamSerializationAllowed = 1; ++n; }
    if (coop) { at[n].id = cudaLaunchAttributeCooperative; at[n].val.cooperative = 1; ++n; }
    cfg.attrs = at; cfg.numAttrs = n;
    HP(2);
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

unsigned long long g_allocGen = 0;   // bumped whenever a workspace buffer moves: cached graphs hold its old address

// grow-only device buffer
struct Buf {
    void* p = nullptr;
    size_t cap = 0;
    cudaError_t need(size_t bytes)
    {
        if (bytes <= cap) return cudaSuccess;
        ++g_allocGen;
        if (p) { cudaFree(p); p = nullptr; cap = 0; }
        size_t want = bytes + bytes / 8 + 256;
        cudaError_t e = cudaMalloc(&p, want);
        if (e != cudaSuccess) { p = nullptr; return e; }
        cap = want;
        return cudaSuccess;
    }
    void release()
    {
        if (p) { cudaFree(p); ++g_allocGen; }
        p = nullptr; cap = 0;
    }
};

// One instantiated CUDA graph of the whole pipeline for one exact set of arguments (pointers included).
struct GraphKey {
    const void *ref, *ev, *out;
    void* ctl;
    GridP g;
    float DD, cutoff, normDose;
    int mode, presort, star, lanes, keyBits, tableMode, algo, statsBins, starLoad;
    long long tableCap;
    const void *statsHist, *statsSummary;
    float statsScale;
    bool operator==(const GraphKey& o) const { return std::memcmp(this, &o, sizeof *this) == 0; }
};
struct GraphEntry {
    GraphKey key;
    cudaGraphExec_t exec = nullptr;
    unsigned long long lastUse = 0;
    int kernels = 0;
};
constexpr int GRAPH_CACHE = 96;    // argument sets x CTL_ROT rotating sets

// One updatable graph per kernel sequence (GraphUpdate): the options that decide WHICH kernels a call launches.
struct UpdKey {
    int star, lanes, algoJu, classes, presort, noNorm;
    bool operator==(const UpdKey& o) const { return std::memcmp(this, &o, sizeof *this) == 0; }
};
struct UpdGraph {
    UpdKey key;
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    cudaGraphNode_t nodes[UPD_MAX_NODES];
    void* funcs[UPD_MAX_NODES];
    int count = 0;
    bool unusable = false;         // this sequence cannot be updated in place (a kernel twice, too many kernels)
    unsigned long long lastUse = 0;
};
constexpr int UPD_CACHE = 4;

// Byte ranges a call in flight reads and writes, for the hazard check of pipelined calls.
struct Span {
    const char *b = nullptr, *e = nullptr;
    void set(const void* p, size_t bytes) { b = static_cast<const char*>(p); e = p ? b + bytes : b; }
    bool hits(const Span& o) const { return b && o.b && b < o.e && o.b < e; }
};
struct CallSpans {
    Span rd[2];   // ref, eval
    Span wr[3];   // out_gamma, stats hist, stats summary
    bool conflicts(const CallSpans& next) const     // `next` starts while this call is still running
    {
        for (const Span& w : wr) {
            for (const Span& r : next.rd) if (w.hits(r)) return true;   // next reads what this call writes
            for (const Span& x : next.wr) if (w.hits(x)) return true;   // both write
        }
        for (const Span& r : rd)
            for (const Span& x : next.wr) if (r.hits(x)) return true;   // next writes what this call reads
        return false;
    }
};

struct Workspace {
    Buf ctl;                       // Ctl[CTL_SLOTS]
    // work lists, `stride` elements each: compacted indices of the evaluated voxels; ring / sorted list (key0, idx0);
    // deep list or sort ping-pong (key1, idx1)
    Buf evalIdx, key0, idx0, key1, idx1;
    long long stride = 0;
    Buf sortK, sortV;              // ping-pong of gamma_sort_pairs (stand-alone)
    Buf tileHist;                  // radix sort
    Buf table, tmpL, tmpIdx;       // offset table: CTL_SLOTS embedded tables, then the large (side-stream) table
    Buf hRef, hEval, hOut;         // device staging of gamma_eval_host
    Buf count;                     // evaluated-voxel count of the two-phase path (large grids)
    cudaEvent_t done = nullptr;    // orders consecutive calls that share this workspace
    bool havePending = false;
    cudaEvent_t stage[7] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};  // opts.profile_stages
    cudaStream_t aux = nullptr;    // side stream: the large offset table is built while k_star runs
    cudaEvent_t evFork = nullptr, evJoin = nullptr;
    void* ctlOwner = nullptr;      // ctl.p the flags below refer to
    bool ctlClean = false;         // the rotating slots are known to be zero / being zeroed by the calls in flight
    int slot = 0;                  // control-block slot of the next call (0 .. CTL_ROT-1)
    unsigned calls = 0;            // calls so far (device timeline)
    void* lastCtl = nullptr;       // control block of the last call
    bool haveStages = false;
    bool stageSort = false, stageTable = false;   // the last profiled call had a sort kernel / a side-stream table
    long long launches = 0;        // kernels launched so far (gamma_launch_count)
    int numSM = 0;
    int occStar[2] = {0, 0};       // resident blocks per SM of k_star<false/true>
    int occTile[2] = {0, 0};       // resident blocks per SM of k_tile_star<false/true>
    int occGeneral = 0;            // resident blocks per SM of k_general_search
    int pdl = -1;                  // programmatic dependent launch between the kernels of a call (GAMMA_PDL=0 disables)
    int graphs = -1;               // replay the call as a cached CUDA graph (GAMMA_GRAPH=0 disables)
    bool frozen = false;           // addresses of this workspace are baked into a caller's CUDA graph: it must not move
    cudaStream_t cap = nullptr;    // capture stream (the caller's may be the legacy default stream, which cannot capture)
    GraphEntry graph[GRAPH_CACHE];
    int numGraphs = 0;
    UpdGraph upd[UPD_CACHE];
    int numUpd = 0;
    unsigned long long graphGen = 0, useClock = 0;
    // keyed graphs hold workspace addresses and go when a buffer moves; the updatable ones get every argument anew with
    // each call and only go with the workspace itself
    void dropGraphs(bool updatableToo = false)
    {
        for (int i = 0; i < numGraphs; ++i)
            if (graph[i].exec) { cudaGraphExecDestroy(graph[i].exec); graph[i].exec = nullptr; }
        numGraphs = 0;
        if (!updatableToo) return;
        for (int i = 0; i < numUpd; ++i) {
            if (upd[i].exec) { cudaGraphExecDestroy(upd[i].exec); upd[i].exec = nullptr; }
            if (upd[i].graph) { cudaGraphDestroy(upd[i].graph); upd[i].graph = nullptr; }
        }
        numUpd = 0;
    }
    // last call, for gamma_get_counters
    cudaStream_t lastStream = nullptr;
    cudaStream_t doneStream = nullptr;   // stream of the last work that used this workspace
    bool chainable = false;              // that work was a pipeline ending in k_table_search (which triggers dependents)
    CallSpans lastSpans;                 // what that pipeline reads and writes
    int lastEarly = 0;                   // the last call started in the tail of its predecessor
    long long numEarly = 0;
    int lastClasses = 0;           // last call used depth classes: list A holds the ring items
    float lastNormDose = 0.0f;     // opts.norm_dose of the last call (0: max(ref) from the control block)
    long long lastN = 0;
    bool haveLast = false;
    size_t bytes() const
    {
        const Buf* all[] = {&ctl, &evalIdx, &key0, &idx0, &key1, &idx1, &sortK, &sortV, &tileHist, &table, &tmpL, &tmpIdx,
                            &hRef, &hEval, &hOut, &count};
        size_t n = 0;
        for (const Buf* b : all) n += b->cap;
        return n;
    }
    void releaseAll()
    {
        Buf* all[] = {&ctl, &evalIdx, &key0, &idx0, &key1, &idx1, &sortK, &sortV, &tileHist, &table, &tmpL, &tmpIdx,
                      &hRef, &hEval, &hOut, &count};
        for (Buf* b : all) b->release();
        if (done) { cudaEventDestroy(done); done = nullptr; }
        for (cudaEvent_t& ev : stage)
            if (ev) { cudaEventDestroy(ev); ev = nullptr; }
        dropGraphs(true);
        if (aux) { cudaStreamDestroy(aux); aux = nullptr; }
        if (cap) { cudaStreamDestroy(cap); cap = nullptr; }
        if (evFork) { cudaEventDestroy(evFork); evFork = nullptr; }
        if (evJoin) { cudaEventDestroy(evJoin); evJoin = nullptr; }
        havePending = false; haveLast = false; haveStages = false; ctlClean = false; ctlOwner = nullptr;
        chainable = false; frozen = false; stride = 0; slot = 0;
        lastSpans = CallSpans();
    }
};

// Workspace 0 serves calls on the caller's stream; 1 .. LANES belong to the library's own lane streams, on which
// back-to-back calls (gamma_opts::back_to_back) and the cases of gamma_eval_batch run so that the kernels of
// consecutive calls overlap on the device; the last one belongs to the calls a caller captures into its own CUDA graph
// (its addresses are baked into that graph, so it never moves once used: gamma_release() is the only way to grow it).
#ifndef GAMMA_LANES
#define GAMMA_LANES 6
#endif
constexpr int LANES = GAMMA_LANES;
constexpr int WS_CAPTURE = 1 + LANES;
Workspace g_pool[2 + LANES];
Workspace* g_cur = &g_pool[0];
Workspace* g_lastWs = &g_pool[0];      // workspace of the last gamma_eval* call (gamma_get_counters)
unsigned g_callNo = 0;                 // gamma_eval* calls so far, all workspaces (device timeline)
#define g_ws (*g_cur)

// Back-to-back calls.  A programmatic dependent that never waits is still not reported complete before its primary
// (measured: profiles/r2_lanes.md), so consecutive calls cannot run ahead of each other on ONE stream.  They are
// spread round-robin over LANES library-owned streams instead, each with its own workspace: the lane waits for what
// was on the caller's stream when the sequence of back-to-back calls began (one event), the caller's stream waits for
// every call (one event per call, so later work of the caller's sees all results), calls on one lane are in stream
// order, and a call that touches a buffer of one of the last B2B_WINDOW - 1 calls on another lane waits for that call.
#ifndef GAMMA_B2B_WINDOW
#define GAMMA_B2B_WINDOW 24
#endif
constexpr int B2B_WINDOW = GAMMA_B2B_WINDOW;   // calls whose buffers are remembered (a multiple of 2 * LANES)
// Back-pressure: every call is also joined into the library's own stream `join`; every B2B_PERIOD calls an event is
// recorded there and the host waits for the event of the period before, so that call j - B2B_WINDOW has ended when call
// j takes over its slot -- one host wait per period instead of one per call.
constexpr int B2B_PERIOD = B2B_WINDOW / 2;
struct LaneState {
    cudaStream_t stream[LANES] = {};
    cudaEvent_t fork = nullptr;
    unsigned long long forkGen = 0, laneFork[LANES] = {};
    bool laneDirty[LANES] = {};        // something other than a library pipeline is the last operation on the lane
    cudaEvent_t done[B2B_WINDOW] = {};
    CallSpans spans[B2B_WINDOW];
    int laneOf[B2B_WINDOW] = {};
    bool used[B2B_WINDOW] = {};
    unsigned long long next = 0;       // number of the next back-to-back call
    cudaStream_t join = nullptr;       // waits for every call; carries the back-pressure events
    cudaEvent_t joined = nullptr;      // recorded on `join` at the start of a period: all earlier calls have ended
    bool haveJoined = false;
    cudaStream_t user = nullptr;       // caller's stream of the sequence in progress
    bool active = false;               // the library's last operation was a back-to-back call on `user`
    bool ready = false;
} g_lanes;

int ensure_device()
{
    if (g_ws.numSM > 0) return GAMMA_OK;
    int dev = 0;
    CU_TRY(cudaGetDevice(&dev));
    int sm = 0;
    CU_TRY(cudaDeviceGetAttribute(&sm, cudaDevAttrMultiProcessorCount, dev));
    g_ws.numSM = sm > 0 ? sm : 148;
    return GAMMA_OK;
}

// host copy of key_digit (common.cuh): the digit of the one-pass presort
int host_key_digit(float key)
{
    unsigned b;
    std::memcpy(&b, &key, 4);
    const int d = (int)(b >> 18) - ((127 - 3) << 5);
    return d < 0 ? 0 : (d > KEY_DIGITS - 1 ? KEY_DIGITS - 1 : d);
}

int order_after_previous(cudaStream_t st)
{
    // Same stream as the last user of the workspace: stream order is enough (and no event sits between the last
    // kernel of that call and the first kernel of this one).  Another stream: wait for the tail of that stream.
    if (!g_ws.done) CU_TRY(cudaEventCreateWithFlags(&g_ws.done, cudaEventDisableTiming));
    if (g_ws.havePending && g_ws.doneStream != st) {
        CU_TRY(cudaEventRecord(g_ws.done, g_ws.doneStream));
        CU_TRY(cudaStreamWaitEvent(st, g_ws.done, 0));
    }
    return GAMMA_OK;
}
int mark_done(cudaStream_t st)
{
    g_ws.doneStream = st;
    g_ws.havePending = true;
    g_ws.chainable = false;
    return GAMMA_OK;
}

// distance from the origin to the triangle (a, b, c) in R^3 (Ericson, Real-Time Collision Detection 5.1.5)
double origin_triangle_distance(const double a[3], const double b[3], const double c[3])
{
    auto dot = [](const double* u, const double* v) { return u[0] * v[0] + u[1] * v[1] + u[2] * v[2]; };
    double ab[3], ac[3], ap[3], bp[3], cp[3], q[3];
    for (int i = 0; i < 3; ++i) { ab[i] = b[i] - a[i]; ac[i] = c[i] - a[i]; ap[i] = -a[i]; bp[i] = -b[i]; cp[i] = -c[i]; }
    const double d1 = dot(ab, ap), d2 = dot(ac, ap);
    auto norm = [&](const double* v) { return std::sqrt(dot(v, v)); };
    if (d1 <= 0 && d2 <= 0) return norm(a);
    const double d3 = dot(ab, bp), d4 = dot(ac, bp);
    if (d3 >= 0 && d4 <= d3) return norm(b);
    const double vc = d1 * d4 - d3 * d2;
    if (vc <= 0 && d1 >= 0 && d3 <= 0) {
        const double t = d1 / (d1 - d3);
        for (int i = 0; i < 3; ++i) q[i] = a[i] + t * ab[i];
        return norm(q);
    }
    const double d5 = dot(ab, cp), d6 = dot(ac, cp);
    if (d6 >= 0 && d5 <= d6) return norm(c);
    const double vb = d5 * d2 - d1 * d6;
    if (vb <= 0 && d2 >= 0 && d6 <= 0) {
        const double t = d2 / (d2 - d6);
        for (int i = 0; i < 3; ++i) q[i] = a[i] + t * ac[i];
        return norm(q);
    }
    const double va = d3 * d6 - d5 * d4;
    if (va <= 0 && (d4 - d3) >= 0 && (d5 - d6) >= 0) {
        const double t = (d4 - d3) / ((d4 - d3) + (d5 - d6));
        for (int i = 0; i < 3; ++i) q[i] = b[i] + t * (c[i] - b[i]);
        return norm(q);
    }
    const double den = 1.0 / (va + vb + vc), v = vb * den, w = vc * den;
    for (int i = 0; i < 3; ++i) q[i] = a[i] + ab[i] * v + ac[i] * w;
    return norm(q);
}

// Distance (in DTA units) from a voxel to the boundary of its star in the Kuhn mesh: the 24 triangles
// opposite the voxel in the 24 tetrahedra that contain it.  Everything outside the star is at least this far.
double star_link_distance(const double h[3])
{
    static const int perms[6][3] = {{0, 1, 2}, {0, 2, 1}, {1, 0, 2}, {1, 2, 0}, {2, 0, 1}, {2, 1, 0}};
    double best = 1e300;
    for (int oc = 0; oc < 8; ++oc) {
        const int o[3] = {(oc & 1) ? -1 : 0, (oc & 2) ? -1 : 0, (oc & 4) ? -1 : 0};
        for (int p = 0; p < 6; ++p) {
            int vtx[4][3];
            for (int a = 0; a < 3; ++a) vtx[0][a] = o[a];
            for (int m = 1; m <= 3; ++m) {
                for (int a = 0; a < 3; ++a) vtx[m][a] = vtx[m - 1][a];
                vtx[m][perms[p][m - 1]] += 1;
            }
            int self = -1;
            for (int m = 0; m <= 3; ++m)
                if (vtx[m][0] == 0 && vtx[m][1] == 0 && vtx[m][2] == 0) self = m;
            if (self < 0) continue;
            double tri[3][3];
            int k = 0;
            for (int m = 0; m <= 3; ++m) {
                if (m == self) continue;
                for (int a = 0; a < 3; ++a) tri[k][a] = vtx[m][a] * h[a];
                ++k;
            }
            const double dist = origin_triangle_distance(tri[0], tri[1], tri[2]);
            if (dist < best) best = dist;
        }
    }
    return best;
}

int make_grid(const int dims[3], const float spacing_mm[3], float DTA_mm, GridP& g)
{
    if (!dims || !spacing_mm) return fail(GAMMA_ERR_INVALID_ARGUMENT, "dims / spacing_mm is NULL");
    if (!(DTA_mm > 0.0f) || !std::isfinite(DTA_mm)) return fail(GAMMA_ERR_INVALID_ARGUMENT, "DTA_mm must be > 0");
    long long N = 1;
    int active = 0;
    for (int a = 0; a < 3; ++a) {
        if (dims[a] < 1) return fail(GAMMA_ERR_INVALID_ARGUMENT, "dims must be >= 1");
        if (!(spacing_mm[a] > 0.0f) || !std::isfinite(spacing_mm[a]))
            return fail(GAMMA_ERR_INVALID_ARGUMENT, "spacing_mm must be > 0");
        N *= dims[a];
        if (N >= (1ll << 31)) return fail(GAMMA_ERR_INVALID_ARGUMENT, "nx*ny*nz must be < 2^31");
        active += dims[a] > 1;
    }
    if (active == 0) return fail(GAMMA_ERR_INVALID_ARGUMENT, "at least one axis must have size > 1");
    // the derived geometry of the last call is kept: a repeated geometry costs a compare, not 48 triangle distances
    struct GeoKey { int d[3]; float s[3]; float dta; };
    static thread_local GeoKey lastKey = {{0, 0, 0}, {0, 0, 0}, 0};
    static thread_local GridP lastGrid;
    GeoKey key;
    std::memset(&key, 0, sizeof key);
    for (int a = 0; a < 3; ++a) { key.d[a] = dims[a]; key.s[a] = spacing_mm[a]; }
    key.dta = DTA_mm;
    if (std::memcmp(&key, &lastKey, sizeof key) == 0) { g = lastGrid; return GAMMA_OK; }
    std::memset(&g, 0, sizeof g);
    double h[3], hh[3];
    for (int a = 0; a < 3; ++a) {
        g.n[a] = dims[a];
        h[a] = dims[a] > 1 ? (double)spacing_mm[a] / (double)DTA_mm : 0.0;
        hh[a] = h[a] * h[a];
        g.h[a] = (float)h[a];
        g.hh[a] = (float)hh[a];
    }
    g.stride[0] = 1; g.stride[1] = dims[0]; g.stride[2] = dims[0] * dims[1];
    g.N = (int)N;
    for (int T = 1; T < 8; ++T) {
        double A = 0.0;
        bool ok = true;
        for (int a = 0; a < 3; ++a)
            if (T & (1 << a)) { ok = ok && h[a] > 0.0; A += hh[a]; }
        g.invA[T] = ok ? (float)(1.0 / A) : 0.0f;
    }
    auto K = [&](int a, int b) { return (hh[a] + hh[b]) > 0.0 ? hh[a] * hh[b] / (hh[a] + hh[b]) : 0.0; };
    g.K3 = (float)K(0, 1); g.K5 = (float)K(0, 2); g.K6 = (float)K(1, 2);
    const double A7 = hh[0] + hh[1] + hh[2];
    g.Kxy7 = (float)(hh[0] * hh[1] / A7); g.Kyz7 = (float)(hh[1] * hh[2] / A7); g.Kzx7 = (float)(hh[2] * hh[0] / A7);
    g.all_active = active == 3;
    {
        double hm = 0.0;
        for (int a = 0; a < 3; ++a)
            if (h[a] > 0.0 && (hm == 0.0 || h[a] < hm)) hm = h[a];
        hm *= (1.0 - 1e-5);
        g.hmin2 = (float)(hm * hm);
        const unsigned dv[2] = {(unsigned)dims[0], (unsigned)dims[0] * (unsigned)dims[1]};
        for (int k = 0; k < 2; ++k) {
            unsigned l = 0;
            while ((1ull << l) < dv[k]) ++l;
            g.divMul[k] = (unsigned)((1ull << (31 + l)) / dv[k] + 1ull);
            g.divSh[k] = 31 + l;
        }
    }
    if (g.all_active) {
        const double rho = star_link_distance(h) * (1.0 - 1e-5);
        g.rho_link2 = (float)(rho * rho);
    }
    lastGrid = g;
    lastKey = key;
    return GAMMA_OK;
}

struct Resolved {
    int presort, star, lanes, keyBits, profile, graph, tableMode, algo, backToBack, starLoad;
    long long tableCap;
    float normDose;
    StatsP stats;      // a6 fused into the gamma kernels (hist == nullptr: off)
};

int resolve_opts(const gamma_opts* o, Resolved& r)
{
    r.presort = 4; r.star = 1; r.lanes = 0; r.keyBits = 16; r.tableCap = 0; r.tableMode = 1; r.normDose = 0.0f;
    r.profile = 0; r.graph = 0; r.algo = 0; r.backToBack = 0; r.starLoad = 0;
    r.stats.hist = nullptr; r.stats.summary = nullptr; r.stats.nbins = 0; r.stats.binScale = 0.0f;
    if (!o) { r.tableCap = TAB_EMBED_MAX_CELLS; return GAMMA_OK; }
    if (o->back_to_back < 0 || o->back_to_back > 1) return fail(GAMMA_ERR_INVALID_ARGUMENT, "opts.back_to_back must be 0 or 1");
    if (o->star_load < 0 || o->star_load > 3) return fail(GAMMA_ERR_INVALID_ARGUMENT, "opts.star_load must be 0, 1, 2 or 3");
    r.starLoad = o->star_load;
    r.backToBack = o->back_to_back;
    if (o->stats_hist || o->stats_summary) {
        if (!o->stats_hist || !o->stats_summary)
            return fail(GAMMA_ERR_INVALID_ARGUMENT, "opts.stats_hist and opts.stats_summary must be given together");
        if (o->stats_nbins < 1 || o->stats_nbins > FUSED_MAX_BINS)
            return fail(GAMMA_ERR_INVALID_ARGUMENT, "opts.stats_nbins must be in [1, 1024] (gamma_stats takes up to 4096)");
        if (!(o->stats_hist_max > 0.0f) || !std::isfinite(o->stats_hist_max))
            return fail(GAMMA_ERR_INVALID_ARGUMENT, "opts.stats_hist_max must be > 0");
        r.stats.hist = o->stats_hist; r.stats.summary = o->stats_summary; r.stats.nbins = o->stats_nbins;
        r.stats.binScale = (float)o->stats_nbins / o->stats_hist_max;
    }
    r.profile = o->profile_stages == 1;
    if (o->graph < 0 || o->graph > 2) return fail(GAMMA_ERR_INVALID_ARGUMENT, "opts.graph must be 0, 1 or 2");
    r.graph = o->graph == 1;
    if (o->presort < 0 || o->presort > 4) return fail(GAMMA_ERR_INVALID_ARGUMENT, "opts.presort must be 0, 1, 2, 3 or 4");
    if (o->star_phase < 0 || o->star_phase > 2) return fail(GAMMA_ERR_INVALID_ARGUMENT, "opts.star_phase must be 0, 1 or 2");
    if (o->presort == 1) r.presort = 1;
    if (o->presort == 2) r.presort = 0;
    if (o->presort == 3) r.presort = 3;
    if (o->star_phase == 2) r.star = 0;
    if (o->lanes_per_voxel != 0) {
        if (o->lanes_per_voxel != 1 && o->lanes_per_voxel != 8 && o->lanes_per_voxel != 32)
            return fail(GAMMA_ERR_INVALID_ARGUMENT, "opts.lanes_per_voxel must be 0, 1, 8 or 32");
        r.lanes = o->lanes_per_voxel;
    }
    if (o->sort_key_bits != 0) {
        if (o->sort_key_bits != 8 && o->sort_key_bits != 16 && o->sort_key_bits != 24 && o->sort_key_bits != 32)
            return fail(GAMMA_ERR_INVALID_ARGUMENT, "opts.sort_key_bits must be 0, 8, 16, 24 or 32");
        r.keyBits = o->sort_key_bits;
    }
    if (o->table_cap != 0) {
        if (o->table_cap < 1 || o->table_cap > (1ll << 26))
            return fail(GAMMA_ERR_INVALID_ARGUMENT, "opts.table_cap must be in [1, 2^26]");
        r.tableCap = o->table_cap;
    }
    if (r.presort == 4 && r.lanes != 0) r.presort = 1;   // depth classes only exist for the adaptive search
    if (o->interpolation < 0 || o->interpolation > 3)
        return fail(GAMMA_ERR_INVALID_ARGUMENT, "opts.interpolation must be 0, 1, 2 or 3");
    if (o->interpolation == 2) { r.algo = 1; r.star = 0; }   // the star phase is interpolation
    if (o->interpolation == 3) { r.algo = 2; r.star = 0; }   // every cell through the table walk and the recursion
    if (o->table_radius < 0 || o->table_radius > 2)
        return fail(GAMMA_ERR_INVALID_ARGUMENT, "opts.table_radius must be 0, 1 or 2");
    if (o->table_radius == 2) r.tableMode = 2;
    if (r.tableCap == 0) r.tableCap = r.tableMode == 1 ? TAB_EMBED_MAX_CELLS : (1ll << 20);
    if (o->norm_dose > 0.0f) r.normDose = o->norm_dose;
    if (std::isnan(o->norm_dose) || std::isinf(o->norm_dose))
        return fail(GAMMA_ERR_INVALID_ARGUMENT, "opts.norm_dose must be finite");
    return GAMMA_OK;
}

int check_criteria(float DD, int mode, float cutoff)
{
    if (!(DD > 0.0f) || !std::isfinite(DD)) return fail(GAMMA_ERR_INVALID_ARGUMENT, "DD must be > 0");
    if (mode != GAMMA_MODE_GLOBAL && mode != GAMMA_MODE_LOCAL) return fail(GAMMA_ERR_INVALID_ARGUMENT, "unknown mode");
    if (!(cutoff >= 0.0f && cutoff < 1.0f)) return fail(GAMMA_ERR_INVALID_ARGUMENT, "low_dose_cutoff must be in [0, 1)");
    return GAMMA_OK;
}

constexpr size_t CTL_BYTES = CTL_SLOTS * sizeof(Ctl);

// ---- TMA descriptors of k_tile_star (tile_star.cuh).  cuTensorMapEncodeTiled is fetched through the runtime (the
// library does not link libcuda); the last few (pointer, dims, box) descriptors are kept.
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn g_encodeTiled = nullptr;
bool g_encodeTried = false;

bool tma_usable(const void* ref, const void* ev, const GridP& g)
{
    if (!g_encodeTried) {
        g_encodeTried = true;
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult q = cudaDriverEntryPointSymbolNotFound;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            g_encodeTiled = reinterpret_cast<EncodeTiledFn>(fn);
        else
            cudaGetLastError();
    }
    return g_encodeTiled != nullptr && g.n[0] % 4 == 0 &&
           ((reinterpret_cast<uintptr_t>(ref) | reinterpret_cast<uintptr_t>(ev)) & 15u) == 0;
}

struct MapKey { const void* p; int n[3]; unsigned box[3]; };
struct MapEntry { MapKey key; CUtensorMap map; unsigned long long use; };
constexpr int MAP_CACHE = 64;
MapEntry g_maps[MAP_CACHE];
int g_numMaps = 0;
unsigned long long g_mapClock = 0;

int tensor_map(const float* p, const GridP& g, unsigned bx, unsigned by, unsigned bz, CUtensorMap& out)
{
    MapKey key;
    std::memset(&key, 0, sizeof key);
    key.p = p; key.n[0] = g.n[0]; key.n[1] = g.n[1]; key.n[2] = g.n[2]; key.box[0] = bx; key.box[1] = by; key.box[2] = bz;
    for (int i = 0; i < g_numMaps; ++i)
        if (std::memcmp(&g_maps[i].key, &key, sizeof key) == 0) { g_maps[i].use = ++g_mapClock; out = g_maps[i].map; return GAMMA_OK; }
    const cuuint64_t dims[3] = {(cuuint64_t)g.n[0], (cuuint64_t)g.n[1], (cuuint64_t)g.n[2]};
    const cuuint64_t strides[2] = {(cuuint64_t)g.n[0] * 4u, (cuuint64_t)g.n[0] * (cuuint64_t)g.n[1] * 4u};
    const cuuint32_t box[3] = {bx, by, bz}, estr[3] = {1, 1, 1};
    CUtensorMap m;
    const CUresult cr = g_encodeTiled(&m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float*>(p), dims, strides, box, estr,
                                      CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                      CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (cr != CUDA_SUCCESS) return fail(GAMMA_ERR_CUDA, "cuTensorMapEncodeTiled failed with code " + std::to_string((int)cr));
    int victim = g_numMaps;
    if (victim == MAP_CACHE) {
        victim = 0;
        for (int i = 1; i < MAP_CACHE; ++i)
            if (g_maps[i].use < g_maps[victim].use) victim = i;
    } else {
        ++g_numMaps;
    }
    g_maps[victim].key = key; g_maps[victim].map = m; g_maps[victim].use = ++g_mapClock;
    out = m;
    return GAMMA_OK;
}

// Grids up to this many voxels get their work lists sized by N; larger grids count their evaluated voxels first (one
// host read of 4 bytes on a call of milliseconds) and get lists sized by M.
constexpr long long LISTS_BY_N_MAX = 1ll << 25;

// Workspace of one call: allocations, side stream, events.  Nothing is allocated once the sizes have been seen.
// `stride`: elements each work list must hold.
int prepare_workspace(const GridP& g, const Resolved& r, long long stride)
{
    int rc = ensure_device();
    if (rc) return rc;
    if (stride < g_ws.stride) stride = g_ws.stride;            // grow-only
    const long long maxTiles = (stride + SORT_TILE - 1) / SORT_TILE;
    const size_t listBytes = (size_t)stride * 4;
    const size_t tableCells = (size_t)CTL_SLOTS * TAB_EMBED_MAX_CELLS + (r.tableCap > TAB_EMBED_MAX_CELLS ? (size_t)r.tableCap : 0);
    if (g_ws.frozen) {
        const bool fits = CTL_BYTES <= g_ws.ctl.cap && listBytes <= g_ws.evalIdx.cap && listBytes <= g_ws.key1.cap &&
                          tableCells * 16 <= g_ws.table.cap && (size_t)r.tableCap * 4 <= g_ws.tmpL.cap &&
                          (r.presort != 3 || (size_t)(maxTiles + 1) * SORT_RADIX * 4 <= g_ws.tileHist.cap);
        if (!fits)
            return fail(GAMMA_ERR_INVALID_ARGUMENT,
                        "this call needs a larger capture workspace, but its addresses are part of a captured CUDA graph; "
                        "call gamma_release() first (that invalidates the captured graphs)");
    }
    CU_TRY(g_ws.ctl.need(CTL_BYTES));
    CU_TRY(g_ws.key0.need(listBytes)); CU_TRY(g_ws.idx0.need(listBytes)); CU_TRY(g_ws.evalIdx.need(listBytes));
    CU_TRY(g_ws.key1.need(listBytes)); CU_TRY(g_ws.idx1.need(listBytes));
    g_ws.stride = stride;
    if (r.presort == 3) CU_TRY(g_ws.tileHist.need((size_t)(maxTiles + 1) * SORT_RADIX * 4));   // + the 256 digit totals
    // the small embedded table exists once per control-block slot (the next call builds its own while this call's
    // search still walks this one); a large table (table_radius 2, table_cap > 1024) lives BEHIND those slots, so a
    // following call's embedded table never aliases it
    CU_TRY(g_ws.table.need(tableCells * 16));
    CU_TRY(g_ws.tmpL.need((size_t)r.tableCap * 4)); CU_TRY(g_ws.tmpIdx.need((size_t)r.tableCap * 4));
    if (!g_ws.aux) {
        CU_TRY(cudaStreamCreateWithFlags(&g_ws.aux, cudaStreamNonBlocking));
        CU_TRY(cudaStreamCreateWithFlags(&g_ws.cap, cudaStreamNonBlocking));
        CU_TRY(cudaEventCreateWithFlags(&g_ws.evFork, cudaEventDisableTiming));
        CU_TRY(cudaEventCreateWithFlags(&g_ws.evJoin, cudaEventDisableTiming));
        CU_TRY(cudaFuncSetAttribute(k_offset_table, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TAB_DYN_SMEM));
    }
    for (int star = 0; star < 2; ++star)
        if (g_ws.occStar[star] == 0) {
            int occ = 0;
            if (star) CU_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_star<true>, STAR_THREADS, 0));
            else CU_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_star<false>, STAR_THREADS, 0));
            g_ws.occStar[star] = occ > 0 ? occ : 1;
        }
    if (g_ws.pdl < 0) {
        const char* env = std::getenv("GAMMA_PDL");
        g_ws.pdl = (env && env[0] == '0') ? 0 : 1;
    }
    if (g_ws.graphs < 0) {
        const char* env = std::getenv("GAMMA_GRAPH");
        g_ws.graphs = (env && env[0] == '0') ? 0 : 1;
    }
    if (r.profile)
        for (cudaEvent_t& evn : g_ws.stage)
            if (!evn) CU_TRY(cudaEventCreate(&evn));
    return GAMMA_OK;
}

// What a call's kernels are told about where they run.
struct CallSlot {
    bool shared;       // the call runs on a lane stream beside the calls of the other lanes: grids that leave room
    int slot;          // control-block / embedded-table slot
    int nextSlot;      // slot k_norm zeroes for the next call (-1: none)
    int waitFirst;     // k_norm waits for the operation in front of it before it reads ref / eval
    bool skipNorm;     // two-phase path: k_norm already ran (and the host has read the evaluated-voxel count)
};

// The kernels of one call on `st` (which may be capturing).  Returns the number of kernels in *launched.
//
//   st :  k_norm -> k_classify -> k_star -> [k_bucket_scatter | LSD radix sort] -> (join) -> k_table_search
//   aux:                    \-> k_offset_table ------------------------------------/     (large tables only)
//
// No memset and no host synchronisation on the path: k_norm zeroes the control block of the next call
// (common.cuh, "Device control block").
int enqueue_kernels(const float* ref, const float* ev, const GridP& g, float DD, int mode, float cutoff,
                    const Resolved& r, float* out, cudaStream_t st, const CallSlot& cs, int* launched)
{
    const long long N = g.N;
    int nk = 0;
    Ctl* base = static_cast<Ctl*>(g_ws.ctl.p);
    Ctl* ctl = base + cs.slot;
    Ctl* next = cs.nextSlot >= 0 ? base + cs.nextSlot : nullptr;
    unsigned *k0 = static_cast<unsigned*>(g_ws.key0.p), *i0 = static_cast<unsigned*>(g_ws.idx0.p);
    unsigned *k1 = static_cast<unsigned*>(g_ws.key1.p), *i1 = static_cast<unsigned*>(g_ws.idx1.p);
    unsigned* e0 = static_cast<unsigned*>(g_ws.evalIdx.p);
    EvalP e;
    e.DD = DD; e.cutoff = cutoff; e.norm_dose = r.normDose; e.mode = mode;
    e.algo = (r.algo == 2 && !g.all_active) ? 0 : r.algo;   // the recursion variant is written for 3D cells
    e.call = g_callNo;
    const int classes = (r.presort == 4 && r.star && g.all_active) ? 1 : 0;   // needs the 3D star phase
    const int presort = (r.presort == 4 && !classes) ? 1 : r.presort;
#define STAGE_MARK(i, s) do { if (r.profile) CU_TRY(cudaEventRecord(g_ws.stage[i], s)); } while (0)
    const int sm = g_ws.numSM;
    const bool pdl = g_ws.pdl != 0;
    // Resident blocks per SM each kernel asks for.  A call on its own gets grids that fill the GPU.  Calls on the lane
    // streams get grids of about half an SM's registers (k_star 4 x 128 x 56 + k_table_search 3 x 128 x 80 = 59 K of
    // 64 K), so that the star phase of one call and the search of another are RESIDENT TOGETHER and fill each other's
    // stalls: every kernel here is latency-bound on its own (issue slots 45 - 50 % busy), and with full-size grids the
    // device timeline shows the kernels of different calls strictly one after the other (profiles/r2_profile.md).
    // GAMMA_LANE_GRIDS=norm,classify,star,search overrides the lane figures (tuning).
    static int laneBlocks[4] = {0, 0, 0, 0};
    if (laneBlocks[0] == 0) {
        laneBlocks[0] = 2; laneBlocks[1] = 4; laneBlocks[2] = 4; laneBlocks[3] = 3;
        if (const char* env = std::getenv("GAMMA_LANE_GRIDS")) {
            int v[4];
            if (std::sscanf(env, "%d,%d,%d,%d", &v[0], &v[1], &v[2], &v[3]) == 4)
                for (int k = 0; k < 4; ++k) if (v[k] >= 1 && v[k] <= 16) laneBlocks[k] = v[k];
        }
    }
    const int normBlocks = cs.shared ? laneBlocks[0] : 4, classifyBlocks = cs.shared ? laneBlocks[1] : 8;
    const int starBlocks = cs.shared ? laneBlocks[2] : 1 << 20, searchBlocks = cs.shared ? laneBlocks[3] : SEARCH_GRID_BLOCKS;
    STAGE_MARK(0, st);
    // a3.  Default: a data-independent PREFIX of the paper's table, as large as table_cap allows; beyond it the search
    // enumerates (exact).  table_radius = 2: the paper's radius max |DD| / dD (A1 steps 1-2), built on a side stream
    // once k_norm's maxima exist.
    // host-side constants of the geometry (table radius / plan, ring constants): kept from the last call
    struct HostGeo { GridP g; long long cap; float radius; TablePlan plan; GammaRingP ring; bool valid; };
    static thread_local HostGeo geo = {};
    const bool geoHit = geo.valid && geo.cap == r.tableCap && std::memcmp(&geo.g, &g, sizeof g) == 0;
    float radius = -1.0f;
    if (r.tableMode == 1 && geoHit) radius = geo.radius;
    else if (r.tableMode == 1) {                           // largest radius whose candidate box has <= cap cells
        float lo = 0.0f, hi = grid_diagonal(g);
        int bx, by, bz;
        if (table_box_cells(g, hi, bx, by, bz) <= r.tableCap) lo = hi;
        else
            for (int it = 0; it < 48; ++it) {
                const float mid = 0.5f * (lo + hi);
                if (table_box_cells(g, mid, bx, by, bz) <= r.tableCap) lo = mid; else hi = mid;
            }
        radius = lo;
    }
    // small prefix tables are built inside k_star, by its first blocks, while they wait for k_classify
    const int embed = (r.tableMode == 1 && r.tableCap <= TAB_EMBED_MAX_CELLS) ? 1 : 0;
    int4* const tabBase = static_cast<int4*>(g_ws.table.p);
    int4* const tab4 = embed ? tabBase + (size_t)cs.slot * (size_t)TAB_EMBED_MAX_CELLS
                             : tabBase + (size_t)CTL_SLOTS * (size_t)TAB_EMBED_MAX_CELLS;
    TablePlan plan;
    std::memset(&plan, 0, sizeof plan);
    if (embed) plan = geoHit ? geo.plan : table_plan_make(g, radius, r.tableCap, 1, TAB_EMBED_BUCKETS);
    auto fork_table = [&]() -> int {
        CU_TRY(cudaEventRecord(g_ws.evFork, st));
        CU_TRY(cudaStreamWaitEvent(g_ws.aux, g_ws.evFork, 0));
        STAGE_MARK(5, g_ws.aux);
        k_offset_table<<<TAB_BLOCKS, TAB_THREADS, TAB_DYN_SMEM, g_ws.aux>>>(
            g, e, ctl, radius, r.tableCap, tab4, static_cast<unsigned*>(g_ws.tmpL.p),
            static_cast<unsigned*>(g_ws.tmpIdx.p), r.tableMode == 1 ? 1 : 0);
        ++nk;
        STAGE_MARK(6, g_ws.aux);
        CU_TRY(cudaEventRecord(g_ws.evJoin, g_ws.aux));
        return GAMMA_OK;
    };
    int rc = GAMMA_OK;
    // a large prefix table needs nothing of this call: forked in front of it (a call with a large table is never
    // started early, so the previous call on the workspace has ended by the time the fork event fires)
    if (r.tableMode == 1 && !embed) { rc = fork_table(); if (rc) return rc; }
    // a0 is not needed at all when the caller gives D_norm and nothing else wants k_norm (its max |DD| sizes the paper's
    // table, it zeroes the fused statistics, the tile kernels read its maxima): the call is then three kernels and
    // k_classify, as its first kernel, takes over the wait and the zeroing of the next control block
    const bool noNorm = !cs.skipNorm && r.normDose > 0.0f && r.tableMode == 1 && r.stats.hist == nullptr &&
                        !(classes && r.starLoad >= 2);
    if (!cs.skipNorm && !noNorm) {                                       // a0 + A1 step 1
        long long blocks = (N + 1023) / 1024;
        int grid = (int)(blocks < 1 ? 1 : (blocks > sm * normBlocks ? sm * normBlocks : blocks));
        CU_TRY(launch_ex(k_norm, grid, NORM_THREADS, 0, st, pdl, false, ref, ev, (int)N, mode, ctl, next, cs.waitFirst,
                         e.call, r.stats, r.tableMode != 1 ? 1 : 0));
        ++nk;
    }
    // a1 + a2 + star phase.  Default: the compacted-list pipeline k_classify -> k_star (doses through L1 / L2).
    // opts.star_load = 2 / 3 (3D grids with depth classes): ONE kernel over spatial tiles, evaluation doses staged by
    // the TMA (tile_star.cuh) or by cooperative loads (what grids whose nx is not a multiple of 4 get anyway).
    // Measured (profiles/r2_star_load.md): the list wins, because every evaluated voxel is in flight at once there,
    // while a block works through its hot tiles one after the other.
    const bool tiles = classes && r.starLoad >= 2;
    if (tiles) {
        STAGE_MARK(1, st);
        if (r.tableMode != 1) { rc = fork_table(); if (rc) return rc; }  // paper's radius: needs k_norm's max |DD|
        const bool tma = r.starLoad != 3 && tma_usable(ref, ev, g);
        CUtensorMap mapRef, mapEv;
        std::memset(&mapRef, 0, sizeof mapRef);
        std::memset(&mapEv, 0, sizeof mapEv);
        if (tma) {
            rc = tensor_map(ref, g, TILE_X, TILE_Y, TILE_Z, mapRef);
            if (rc) return rc;
            rc = tensor_map(ev, g, HALO_PX, HALO_Y, HALO_Z, mapEv);
            if (rc) return rc;
        }
        TileGrid tg;
        tg.tx = (g.n[0] + TILE_X - 1) / TILE_X; tg.ty = (g.n[1] + TILE_Y - 1) / TILE_Y; tg.tz = (g.n[2] + TILE_Z - 1) / TILE_Z;
        const unsigned dv[2] = {(unsigned)tg.tx, (unsigned)tg.tx * (unsigned)tg.ty};
        for (int k = 0; k < 2; ++k) {
            unsigned l = 0;
            while ((1ull << l) < dv[k]) ++l;
            tg.divMul[k] = (unsigned)((1ull << (31 + l)) / dv[k] + 1ull);
            tg.divSh[k] = 31 + l;
        }
        const long long numTiles = (long long)tg.tx * tg.ty * tg.tz;
        if (g_ws.occTile[tma] == 0) {
            int occ = 0;
            if (tma) CU_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_tile_star<true>, TILE_VOX, 0));
            else CU_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_tile_star<false>, TILE_VOX, 0));
            g_ws.occTile[tma] = occ > 0 ? occ : 1;
        }
        const long long resident = (long long)sm * g_ws.occTile[tma];
        const int grid = (int)(numTiles > resident ? resident : numTiles);
        unsigned *tabL = static_cast<unsigned*>(g_ws.tmpL.p), *tabI = static_cast<unsigned*>(g_ws.tmpIdx.p);
        if (tma)
            CU_TRY(launch_ex(k_tile_star<true>, grid, TILE_VOX, 0, st, pdl, false, mapRef, mapEv, ref, ev, out, g, e, ctl, k0, i0,
                             k1, i1, embed, plan, tab4, tabL, tabI, r.stats, tg));
        else
            CU_TRY(launch_ex(k_tile_star<false>, grid, TILE_VOX, 0, st, pdl, false, mapRef, mapEv, ref, ev, out, g, e, ctl, k0, i0,
                             k1, i1, embed, plan, tab4, tabL, tabI, r.stats, tg));
        ++nk;
    } else {
    {                                                                    // a1: exclusion + compaction
        long long chunks = (N + PREP_CHUNK - 1) / PREP_CHUNK;
        int grid = (int)(chunks > sm * classifyBlocks ? sm * classifyBlocks : chunks);
        CU_TRY(launch_ex(k_classify, grid, PREP_THREADS, 0, st, pdl, false, ref, out, g, e, ctl, e0, r.stats,
                         noNorm ? next : static_cast<Ctl*>(nullptr), noNorm ? 1 : 0));
        ++nk;
    }
    STAGE_MARK(1, st);
    if (r.tableMode != 1) { rc = fork_table(); if (rc) return rc; }      // paper's radius: needs k_norm's max |DD|
    {                                                                    // star phase over the compacted voxels
        unsigned *tabL = static_cast<unsigned*>(g_ws.tmpL.p), *tabI = static_cast<unsigned*>(g_ws.tmpIdx.p);
        long long warps = (N + 31) / 32, blocks = (warps + STAR_THREADS / 32 - 1) / (STAR_THREADS / 32);
        const long long resident = (long long)sm * (g_ws.occStar[r.star] < starBlocks ? g_ws.occStar[r.star] : starBlocks);
        int grid = (int)(blocks > resident ? resident : blocks);
        if (r.star)
            CU_TRY(launch_ex(k_star<true>, grid, STAR_THREADS, 0, st, pdl, false, ref, ev, out, g, e, ctl, e0, k0, i0, k1, i1, classes,
                             embed, plan, tab4, tabL, tabI, r.stats));
        else
            CU_TRY(launch_ex(k_star<false>, grid, STAR_THREADS, 0, st, pdl, false, ref, ev, out, g, e, ctl, e0, k0, i0, k1, i1, classes,
                             embed, plan, tab4, tabL, tabI, r.stats));
        ++nk;
    }
    }
    STAGE_MARK(2, st);
    if (!embed) CU_TRY(cudaStreamWaitEvent(st, g_ws.evJoin, 0));   // before the presort: presort -> search stay adjacent
    g_ws.stageTable = !embed;
    g_ws.stageSort = presort == 1 || presort == 3;    // no sort kernel: no event either (sort_ms = 0, not a gap)
    const unsigned *lk = k0, *li = i0;
    if (presort == 1) {                                                // a2: one-pass MSD bucket presort
        CU_TRY(launch_ex(k_bucket_scatter, sm * 2, SCATTER_THREADS, 0, st, pdl, false, ctl, k0, i0, k1, i1));
        ++nk;
        lk = k1; li = i1;
    } else if (presort == 3) {                                         // a2: full LSD radix sort of the keys
        int where = radix_sort_enqueue(k0, i0, k1, i1, &ctl->nSearch, g_ws.stride, 32 - r.keyBits, 32,
                                       static_cast<unsigned*>(g_ws.tileHist.p), st);
        nk += 3 * (r.keyBits / 8);
        if (where) { lk = k1; li = i1; }
    }
    if (g_ws.stageSort) STAGE_MARK(3, st);
    {                                                                    // a4 + a5
        const int grid = sm * (r.lanes == 0 ? searchBlocks : 4 * (256 / SEARCH_THREADS));   // resident blocks
        const int4* tab = tab4;
        // adaptive lanes: an item is "deep" when its key exceeds the smallest non-zero table distance
        float hmin = 0.0f;
        for (int a = 0; a < 3; ++a)
            if (g.h[a] > 0.0f && (hmin == 0.0f || g.h[a] < hmin)) hmin = g.h[a];
        const int deepDigit = (presort == 1 || presort == 3) ? host_key_digit(hmin) + 1 : KEY_DIGITS;
        GammaRingP ring;
        std::memset(&ring, 0, sizeof ring);
        if (classes && geoHit) {
            ring = geo.ring;
        } else if (classes) {
            const double hh[3] = {(double)g.h[0] * g.h[0], (double)g.h[1] * g.h[1], (double)g.h[2] * g.h[2]};
            gamma_ring_constants(hh, ring);
        }
        if (!geoHit && r.tableMode == 1 && g.all_active && classes) {
            geo.g = g; geo.cap = r.tableCap; geo.radius = radius; geo.plan = plan; geo.ring = ring; geo.valid = true;
        }
#define LAUNCH_SEARCH(...) CU_TRY(launch_ex(k_table_search<__VA_ARGS__>, grid, SEARCH_THREADS, 0, st, pdl, false, ref, ev, out, g, e, \
                                            ctl, lk, li, k1, i1, tab, deepDigit, classes, ring, r.stats))
        if (e.algo == 2 && r.lanes == 1) LAUNCH_SEARCH(1, true);
        else if (e.algo == 2) LAUNCH_SEARCH(0, true);
        else if (r.lanes == 1) LAUNCH_SEARCH(1);
        else if (r.lanes == 8) LAUNCH_SEARCH(8);
        else if (r.lanes == 32) LAUNCH_SEARCH(32);
        else LAUNCH_SEARCH(0);
#undef LAUNCH_SEARCH
        ++nk;
    }
    STAGE_MARK(4, st);
#undef STAGE_MARK
    *launched = nk;
    g_ws.lastClasses = classes;
    g_ws.lastNormDose = r.normDose;
    g_ws.lastCtl = ctl;
    return GAMMA_OK;
}

// Count of the evaluated voxels for the two-phase path of large grids (same decision as k_classify).
__global__ void __launch_bounds__(256)
k_count_eval(const float* __restrict__ ref, int N, EvalP e, const Ctl* __restrict__ ctl, unsigned* __restrict__ count)
{
    const float dnormF = e.norm_dose > 0.0f ? e.norm_dose : ordered_to_float(ctl->normOrd);
    const double dnorm = (double)dnormF;
    const float thrUp = __double2float_ru((double)e.cutoff * dnorm);     // same decision as k_classify
    const bool globalOk = (double)e.DD * dnorm > 0.0;
    unsigned c = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
        const float Dr = __ldg(ref + i);
        const bool excluded = (Dr < thrUp) || (e.mode == 0 ? !globalOk : !(Dr > 0.0f));
        c += excluded ? 0u : 1u;
    }
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) c += __shfl_xor_sync(0xffffffffu, c, s);
    if ((threadIdx.x & 31) == 0 && c) atomicAdd(count, c);
}

// The rotating control blocks exist and are zero where nothing is in flight; after a call that failed half-way nothing
// is known about them: zero them behind whatever is still running.
int ensure_ctl(cudaStream_t st)
{
    if (g_ws.ctl.p && g_ws.ctl.p == g_ws.ctlOwner && g_ws.ctlClean) return GAMMA_OK;
    CU_TRY(g_ws.ctl.need(CTL_BYTES));
    CU_TRY(cudaMemsetAsync(g_ws.ctl.p, 0, CTL_BYTES, st));
    g_ws.ctlOwner = g_ws.ctl.p;
    g_ws.ctlClean = true;
    g_ws.slot = 0;
    g_ws.chainable = false;
    return GAMMA_OK;
}

// Enqueue the whole hot path on `st` (device pointers) with the current workspace.  Caller holds g_mu.
//
// allowEarly: `st` is a library-owned lane stream whose last operation is the previous pipeline of this workspace:
// k_norm may then start in the tail of that call (it is launched as a programmatic dependent of its k_table_search,
// reads this call's inputs only and ends after that call).  On a caller's stream the first kernel always waits for the
// operation in front of it: the library cannot see what that operation is.
//
// opts.graph = 1: a call with arguments seen before (same pointers, geometry, criteria, options, slot) replays a cached
// CUDA graph of its kernels.  A stream that the CALLER is capturing gets the kernels as nodes of the caller's graph, on
// the capture workspace.
int enqueue_pipeline(const float* ref, const float* ev, const GridP& g, float DD, int mode, float cutoff,
                     const Resolved& r, float* out, cudaStream_t st, bool allowEarly, bool shared = false)
{
    cudaStreamCaptureStatus capStatus = cudaStreamCaptureStatusNone;
    if (!allowEarly) CU_TRY(cudaStreamIsCapturing(st, &capStatus));      // lane streams are never captured
    const bool capturing = capStatus != cudaStreamCaptureStatusNone;
    const long long N = g.N;
    int rc;
    if (capturing) {
        // The kernels become nodes of the caller's graph.  The call must be self-contained (its replays do not pass
        // through this function): its own workspace (never moved afterwards), its own control block cleared by a
        // memset node; ordering against other work is the captured stream's.
        Workspace* keep = g_cur;
        g_cur = &g_pool[WS_CAPTURE];
        {   // cudaMalloc is not a stream operation, but a capture in "global" mode forbids it: relax for the allocation
            cudaStreamCaptureMode cm = cudaStreamCaptureModeRelaxed;
            cudaThreadExchangeStreamCaptureMode(&cm);
            rc = prepare_workspace(g, r, N);
            cudaThreadExchangeStreamCaptureMode(&cm);
        }
        int launched = 0;
        if (rc == GAMMA_OK) {
            g_ws.frozen = true;
            Ctl* ctl = static_cast<Ctl*>(g_ws.ctl.p) + CTL_CAPTURE;
            cudaError_t ce = cudaMemsetAsync(ctl, 0, sizeof(Ctl), st);
            if (ce != cudaSuccess) rc = fail(GAMMA_ERR_CUDA, std::string("cudaMemsetAsync: ") + cudaGetErrorString(ce));
        }
        if (rc == GAMMA_OK) {
            Resolved rr = r;
            rr.profile = 0;
            CallSlot cs;
            cs.slot = CTL_CAPTURE; cs.nextSlot = -1; cs.waitFirst = 1; cs.skipNorm = false; cs.shared = false;
            rc = enqueue_kernels(ref, ev, g, DD, mode, cutoff, rr, out, st, cs, &launched);
        }
        if (rc == GAMMA_OK) {
            g_ws.launches += launched;
            g_ws.haveStages = false;
            g_ws.lastStream = nullptr; g_ws.lastN = g.N; g_ws.haveLast = true; g_ws.lastEarly = 0;
            g_lastWs = g_cur;
        }
        g_cur = keep;
        return rc;
    }
    long long byNMax = LISTS_BY_N_MAX;
    { HP(6); if (const char* env = std::getenv("GAMMA_LISTS_BY_N_MAX")) byNMax = std::atoll(env); }  // tests: two-phase path on small grids
    const bool twoPhase = N > byNMax;
    const bool useGraph = g_ws.graphs != 0 && r.graph && !r.profile && !twoPhase;
    {
        HP(4);
        rc = ensure_device();
        if (rc) return rc;
        rc = order_after_previous(st);
        if (rc) return rc;
        rc = ensure_ctl(st);
        if (rc) return rc;
    }
    g_ws.ctlClean = false;                                 // set again when everything below was enqueued
    CallSlot cs;
    cs.slot = g_ws.slot;
    cs.nextSlot = (g_ws.slot + 1) % CTL_ROT;
    cs.skipNorm = false;
    cs.shared = shared;
    long long stride = N;
    if (twoPhase) {
        // a0, then the count of evaluated voxels, read by the host: the lists are sized by M
        CU_TRY(g_ws.count.need(16));
        Ctl* base = static_cast<Ctl*>(g_ws.ctl.p);
        EvalP e0p;
        e0p.DD = DD; e0p.cutoff = cutoff; e0p.norm_dose = r.normDose; e0p.mode = mode; e0p.algo = 0; e0p.call = g_callNo;
        CU_TRY(cudaMemsetAsync(g_ws.count.p, 0, 16, st));
        const int sm = g_ws.numSM;
        CU_TRY(launch_ex(k_norm, sm * 4, NORM_THREADS, 0, st, false, false, ref, ev, (int)N, mode, base + cs.slot,
                         base + cs.nextSlot, 1, g_callNo, r.stats, r.tableMode != 1 ? 1 : 0));
        k_count_eval<<<sm * 8, 256, 0, st>>>(ref, (int)N, e0p, base + cs.slot, static_cast<unsigned*>(g_ws.count.p));
        unsigned M = 0;
        CU_TRY(cudaMemcpyAsync(&M, g_ws.count.p, 4, cudaMemcpyDeviceToHost, st));
        CU_TRY(cudaStreamSynchronize(st));
        g_ws.launches += 2;
        stride = (long long)M + 1024;
        cs.skipNorm = true;
    }
    { HP(4); rc = prepare_workspace(g, r, stride); }
    if (rc) return rc;
    // ---- may k_norm start in the tail of the previous call?
    CallSpans mine;
    const size_t bytes = (size_t)N * 4;
    mine.rd[0].set(ref, bytes); mine.rd[1].set(ev, bytes); mine.wr[0].set(out, bytes);
    mine.wr[1].set(r.stats.hist, (size_t)r.stats.nbins * 8); mine.wr[2].set(r.stats.summary, sizeof(gamma_summary));
    static const bool overlapCalls = !(std::getenv("GAMMA_OVERLAP_CALLS") && std::getenv("GAMMA_OVERLAP_CALLS")[0] == '0');
    const bool embed = r.tableMode == 1 && r.tableCap <= TAB_EMBED_MAX_CELLS;
    // Calls on a lane stream (and opts.graph = 1 calls) go out as ONE graph launch whose kernel nodes get this call's
    // arguments (GraphUpdate): 4 x 0.4 us + 1.3 us of host time instead of 4 x 3.3 us.  Only for kernel sequences without
    // side stream, events or repeated kernels; everything else is launched kernel by kernel.
    static const bool updGraphs = !(std::getenv("GAMMA_UPDATE_GRAPHS") && std::getenv("GAMMA_UPDATE_GRAPHS")[0] == '0');
    bool useUpd = updGraphs && g_ws.graphs != 0 && (shared || r.graph) && !r.profile && !twoPhase && embed &&
                  r.starLoad <= 1 && r.presort != 3;
    const bool early = allowEarly && overlapCalls && g_ws.pdl != 0 && g_ws.chainable && g_ws.havePending &&
                       g_ws.doneStream == st && !r.profile && !useGraph && !useUpd && !twoPhase && embed &&
                       !g_ws.lastSpans.conflicts(mine);
    cs.waitFirst = early ? 0 : 1;
    g_ws.haveStages = false;

    int launched = 0;
    bool launchedByUpdate = false;
    if (useUpd) {
        UpdKey uk;
        std::memset(&uk, 0, sizeof uk);
        uk.star = r.star; uk.lanes = r.lanes; uk.algoJu = r.algo == 2; uk.classes = g.all_active; uk.presort = r.presort;
        uk.noNorm = r.normDose > 0.0f && r.stats.hist == nullptr;
        UpdGraph* hit = nullptr;
        for (int i = 0; i < g_ws.numUpd; ++i)
            if (g_ws.upd[i].key == uk) { hit = &g_ws.upd[i]; break; }
        if (!hit) {                                        // build: capture this call once, keep graph, exec and nodes
            int victim = 0;                                // a free entry, else the least recently used one
            if (g_ws.numUpd < UPD_CACHE) victim = g_ws.numUpd++;
            else
                for (int i = 1; i < UPD_CACHE; ++i)
                    if (g_ws.upd[i].lastUse < g_ws.upd[victim].lastUse) victim = i;
            UpdGraph& ug = g_ws.upd[victim];
            if (ug.exec) { cudaGraphExecDestroy(ug.exec); ug.exec = nullptr; }
            if (ug.graph) { cudaGraphDestroy(ug.graph); ug.graph = nullptr; }
            ug.key = uk; ug.count = 0; ug.unusable = false;
            LaunchRecord rec;
            std::memset(&rec, 0, sizeof rec);
            CU_TRY(cudaStreamBeginCapture(g_ws.cap, cudaStreamCaptureModeThreadLocal));
            g_rec = &rec;
            rc = enqueue_kernels(ref, ev, g, DD, mode, cutoff, r, out, g_ws.cap, cs, &launched);
            g_rec = nullptr;
            cudaError_t ce = cudaStreamEndCapture(g_ws.cap, &ug.graph);
            if (rc) { if (ug.graph) { cudaGraphDestroy(ug.graph); ug.graph = nullptr; } ug.unusable = true; return rc; }
            if (ce != cudaSuccess) { ug.unusable = true; return fail(GAMMA_ERR_CUDA, std::string("cudaStreamEndCapture: ") + cudaGetErrorString(ce)); }
            ug.unusable = rec.overflow || rec.count == 0;
            for (int a = 0; a < rec.count && !ug.unusable; ++a)
                for (int b = a + 1; b < rec.count; ++b)
                    if (rec.funcs[a] == rec.funcs[b]) ug.unusable = true;       // a node is found by its kernel
            if (!ug.unusable) {
                cudaGraphNode_t all[4 * UPD_MAX_NODES];
                size_t nAll = 0;
                CU_TRY(cudaGraphGetNodes(ug.graph, nullptr, &nAll));
                if (nAll > 4 * UPD_MAX_NODES) ug.unusable = true;
                else CU_TRY(cudaGraphGetNodes(ug.graph, all, &nAll));
                for (int a = 0; a < rec.count && !ug.unusable; ++a) {
                    bool found = false;
                    for (size_t i = 0; i < nAll && !found; ++i) {
                        cudaGraphNodeType ty;
                        CU_TRY(cudaGraphNodeGetType(all[i], &ty));
                        if (ty != cudaGraphNodeTypeKernel) continue;
                        cudaKernelNodeParams kp;
                        CU_TRY(cudaGraphKernelNodeGetParams(all[i], &kp));
                        if (kp.func == rec.funcs[a]) { ug.nodes[a] = all[i]; ug.funcs[a] = rec.funcs[a]; found = true; }
                    }
                    if (!found) ug.unusable = true;
                }
                ug.count = rec.count;
            }
            if (!ug.unusable) {
                ce = cudaGraphInstantiate(&ug.exec, ug.graph, 0);
                if (ce != cudaSuccess) { ug.unusable = true; cudaGetLastError(); }
            }
            hit = &ug;
        }
        hit->lastUse = ++g_ws.useClock;
        if (!hit->unusable) {
            GraphUpdate u = {hit->exec, hit->nodes, hit->funcs, hit->count, 0, true};
            g_upd = &u;
            rc = enqueue_kernels(ref, ev, g, DD, mode, cutoff, r, out, st, cs, &launched);
            g_upd = nullptr;
            if (rc) return rc;
            if (u.ok && u.idx == u.count) {
                HP(9);
                CU_TRY(cudaGraphLaunch(hit->exec, st));
                launchedByUpdate = true;
            } else {
                hit->unusable = true;                      // not the kernels the graph was built from: launch them one by one
            }
        }
    }
    if (launchedByUpdate) {
    } else if (!useGraph) {
        HP(7);
        rc = enqueue_kernels(ref, ev, g, DD, mode, cutoff, r, out, st, cs, &launched);
        if (rc) return rc;
    } else {
        if (g_ws.graphGen != g_allocGen) { g_ws.dropGraphs(); g_ws.graphGen = g_allocGen; }
        Ctl* ctl = static_cast<Ctl*>(g_ws.ctl.p) + cs.slot;
        GraphKey key;
        std::memset(&key, 0, sizeof key);
        key.ref = ref; key.ev = ev; key.out = out; key.ctl = ctl; key.g = g;
        key.DD = DD; key.cutoff = cutoff; key.normDose = r.normDose;
        key.mode = mode; key.presort = r.presort; key.star = r.star; key.lanes = r.lanes; key.keyBits = r.keyBits;
        key.tableCap = r.tableCap; key.tableMode = r.tableMode; key.algo = r.algo;
        key.statsHist = r.stats.hist; key.statsSummary = r.stats.summary; key.statsBins = r.stats.nbins;
        key.statsScale = r.stats.binScale; key.starLoad = r.starLoad;
        GraphEntry* hit = nullptr;
        for (int i = 0; i < g_ws.numGraphs; ++i)
            if (g_ws.graph[i].key == key) { hit = &g_ws.graph[i]; break; }
        if (!hit) {
            cudaGraph_t graph = nullptr;
            CU_TRY(cudaStreamBeginCapture(g_ws.cap, cudaStreamCaptureModeThreadLocal));
            rc = enqueue_kernels(ref, ev, g, DD, mode, cutoff, r, out, g_ws.cap, cs, &launched);
            cudaError_t ce = cudaStreamEndCapture(g_ws.cap, &graph);
            if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
            if (ce != cudaSuccess) return fail(GAMMA_ERR_CUDA, std::string("cudaStreamEndCapture: ") + cudaGetErrorString(ce));
            cudaGraphExec_t exec = nullptr;
            ce = cudaGraphInstantiate(&exec, graph, 0);
            cudaGraphDestroy(graph);
            if (ce != cudaSuccess) return fail(GAMMA_ERR_CUDA, std::string("cudaGraphInstantiate: ") + cudaGetErrorString(ce));
            int victim = g_ws.numGraphs;
            if (victim == GRAPH_CACHE) {                   // evict the least recently used
                victim = 0;
                for (int i = 1; i < GRAPH_CACHE; ++i)
                    if (g_ws.graph[i].lastUse < g_ws.graph[victim].lastUse) victim = i;
                cudaGraphExecDestroy(g_ws.graph[victim].exec);
            } else {
                ++g_ws.numGraphs;
            }
            hit = &g_ws.graph[victim];
            hit->key = key; hit->exec = exec; hit->kernels = launched;
        }
        hit->lastUse = ++g_ws.useClock;
        launched = hit->kernels;
        g_ws.lastCtl = ctl;
        CU_TRY(cudaGraphLaunch(hit->exec, st));
    }
    g_ws.launches += launched;
    g_ws.haveStages = r.profile != 0 && !useGraph;
    CU_TRY(cudaGetLastError());
    rc = mark_done(st);
    if (rc) return rc;
    g_ws.chainable = true;
    g_ws.lastSpans = mine;
    g_ws.slot = (g_ws.slot + 1) % CTL_ROT;
    ++g_ws.calls;
    ++g_callNo;
    g_ws.ctlClean = true;
    g_ws.lastStream = st; g_ws.lastN = g.N; g_ws.haveLast = true;
    // (a call without k_norm starts with a k_classify that waits for its predecessor at its top: not an early start)
    const bool startedEarly = early && !(r.normDose > 0.0f && r.tableMode == 1 && r.stats.hist == nullptr && r.starLoad <= 1);
    g_ws.lastEarly = startedEarly ? 1 : 0;
    g_ws.numEarly += startedEarly ? 1 : 0;
    g_lastWs = g_cur;
    return GAMMA_OK;
}

int lanes_init()
{
    if (g_lanes.ready) return GAMMA_OK;
    CU_TRY(cudaEventCreateWithFlags(&g_lanes.fork, cudaEventDisableTiming));
    for (int l = 0; l < LANES; ++l) CU_TRY(cudaStreamCreateWithFlags(&g_lanes.stream[l], cudaStreamNonBlocking));
    for (int w = 0; w < B2B_WINDOW; ++w) CU_TRY(cudaEventCreateWithFlags(&g_lanes.done[w], cudaEventDisableTiming));
    CU_TRY(cudaStreamCreateWithFlags(&g_lanes.join, cudaStreamNonBlocking));
    CU_TRY(cudaEventCreateWithFlags(&g_lanes.joined, cudaEventDisableTiming));
    g_lanes.ready = true;
    return GAMMA_OK;
}

// One back-to-back call (see LaneState).  `fresh`: the sequence starts here -- the lanes wait for what is on `user` now.
int enqueue_on_lane(const float* ref, const float* ev, const GridP& g, float DD, int mode, float cutoff,
                    const Resolved& r, float* out, cudaStream_t user, bool fresh)
{
    int rc = lanes_init();
    if (rc) return rc;
    LaneState& L = g_lanes;
    if (fresh || !L.active || L.user != user) {
        CU_TRY(cudaEventRecord(L.fork, user));
        ++L.forkGen;
        L.user = user;
    }
    L.active = false;                                      // set again on success
    const unsigned long long j = L.next;
    const int w = (int)(j % B2B_WINDOW), lane = (int)(j % LANES);
    if (j % B2B_PERIOD == 0) {                             // back-pressure: calls up to j - B2B_PERIOD - 1 have ended
        HP(1);
        if (L.haveJoined) CU_TRY(cudaEventSynchronize(L.joined));
        CU_TRY(cudaEventRecord(L.joined, L.join));         // covers every call before this one
        L.haveJoined = true;
    }
    cudaStream_t st = L.stream[lane];
    if (L.laneFork[lane] != L.forkGen) {
        CU_TRY(cudaStreamWaitEvent(st, L.fork, 0));
        L.laneFork[lane] = L.forkGen;
        L.laneDirty[lane] = true;
    }
    CallSpans mine;
    const size_t bytes = (size_t)g.N * 4;
    mine.rd[0].set(ref, bytes); mine.rd[1].set(ev, bytes); mine.wr[0].set(out, bytes);
    mine.wr[1].set(r.stats.hist, (size_t)r.stats.nbins * 8); mine.wr[2].set(r.stats.summary, sizeof(gamma_summary));
    for (int back = 1; back < B2B_WINDOW && (unsigned long long)back <= j; ++back) {
        const int wi = (int)((j - back) % B2B_WINDOW);
        if (L.used[wi] && L.laneOf[wi] != lane && L.spans[wi].conflicts(mine)) {
            CU_TRY(cudaStreamWaitEvent(st, L.done[wi], 0));           // that call writes what this one touches, or reads what it writes
            L.laneDirty[lane] = true;
        }
    }
    Workspace* keep = g_cur;
    g_cur = &g_pool[1 + lane];
    rc = enqueue_pipeline(ref, ev, g, DD, mode, cutoff, r, out, st, !L.laneDirty[lane], true);
    g_cur = keep;
    if (rc) { L.laneDirty[lane] = true; return rc; }
    L.laneDirty[lane] = false;
    {
        HP(3);
        CU_TRY(cudaEventRecord(L.done[w], st));
        CU_TRY(cudaStreamWaitEvent(user, L.done[w], 0));              // the caller's stream sees the result
        CU_TRY(cudaStreamWaitEvent(L.join, L.done[w], 0));
    }
    L.spans[w] = mine; L.laneOf[w] = lane; L.used[w] = true;
    ++L.next;
    L.active = true;
    return GAMMA_OK;
}

// gamma_eval_host_batch: copy engines and compute overlapped.  Three sets of device staging buffers rotate; the
// host-to-device copies run on one library stream, the kernels on lane 0, the device-to-host copies on another stream.
constexpr int HB_DEPTH = 3;
struct HostBatchState {
    Buf ref[HB_DEPTH], ev[HB_DEPTH], out[HB_DEPTH];
    cudaStream_t h2d = nullptr, d2h = nullptr;
    cudaEvent_t start = nullptr, copied[HB_DEPTH] = {}, computed[HB_DEPTH] = {}, freed[HB_DEPTH] = {};
    bool ready = false;
    void release()
    {
        for (int k = 0; k < HB_DEPTH; ++k) {
            ref[k].release(); ev[k].release(); out[k].release();
            if (copied[k]) { cudaEventDestroy(copied[k]); copied[k] = nullptr; }
            if (computed[k]) { cudaEventDestroy(computed[k]); computed[k] = nullptr; }
            if (freed[k]) { cudaEventDestroy(freed[k]); freed[k] = nullptr; }
        }
        if (start) { cudaEventDestroy(start); start = nullptr; }
        if (h2d) { cudaStreamDestroy(h2d); h2d = nullptr; }
        if (d2h) { cudaStreamDestroy(d2h); d2h = nullptr; }
        ready = false;
    }
} g_hb;

// any other library operation ends a sequence of back-to-back calls: the next one forks from the caller's stream again
void end_b2b_sequence() { g_lanes.active = false; }

}  // namespace

extern "C" {

int gamma_eval_ex(const float* ref, const float* eval, const int dims[3], const float spacing_mm[3], float DD,
                  float DTA_mm, int mode, float low_dose_cutoff, const gamma_opts* opts, float* out_gamma,
                  void* stream)
{
    HP(0);
    g_err.clear();
    if (!ref || !eval || !out_gamma) return fail(GAMMA_ERR_INVALID_ARGUMENT, "ref / eval / out_gamma is NULL");
    GridP g;
    Resolved r;
    int rc;
    {
        HP(5);
        rc = make_grid(dims, spacing_mm, DTA_mm, g);
        if (rc) return rc;
        rc = check_criteria(DD, mode, low_dose_cutoff);
        if (rc) return rc;
        rc = resolve_opts(opts, r);
        if (rc) return rc;
    }
    std::lock_guard<std::mutex> lock(g_mu);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (r.backToBack) {
        // honoured for the default kind of call only; everything else runs on the caller's stream, in stream order
        cudaStreamCaptureStatus capStatus = cudaStreamCaptureStatusNone;
        CU_TRY(cudaStreamIsCapturing(st, &capStatus));
        long long byNMax = LISTS_BY_N_MAX;
        if (const char* env = std::getenv("GAMMA_LISTS_BY_N_MAX")) byNMax = std::atoll(env);
        static const bool overlapCalls = !(std::getenv("GAMMA_OVERLAP_CALLS") && std::getenv("GAMMA_OVERLAP_CALLS")[0] == '0');
        if (overlapCalls && capStatus == cudaStreamCaptureStatusNone && !r.profile && !r.graph && g.N <= byNMax &&
            r.tableMode == 1 && r.tableCap <= TAB_EMBED_MAX_CELLS)
            return enqueue_on_lane(ref, eval, g, DD, mode, low_dose_cutoff, r, out_gamma, st, false);
    }
    end_b2b_sequence();
    return enqueue_pipeline(ref, eval, g, DD, mode, low_dose_cutoff, r, out_gamma, st, false);
}

int gamma_eval(const float* ref, const float* eval, const int dims[3], const float spacing_mm[3], float DD,
               float DTA_mm, int mode, float low_dose_cutoff, float* out_gamma, void* stream)
{
    return gamma_eval_ex(ref, eval, dims, spacing_mm, DD, DTA_mm, mode, low_dose_cutoff, nullptr, out_gamma, stream);
}

int gamma_eval_batch(int n_cases, const float* const* ref, const float* const* eval, const int* dims,
                     const float* spacing_mm, float DD, float DTA_mm, int mode, float low_dose_cutoff,
                     const gamma_opts* opts, float* const* out_gamma, void* stream)
{
    g_err.clear();
    if (n_cases < 0) return fail(GAMMA_ERR_INVALID_ARGUMENT, "n_cases must be >= 0");
    if (n_cases == 0) return GAMMA_OK;
    if (!ref || !eval || !out_gamma || !dims || !spacing_mm)
        return fail(GAMMA_ERR_INVALID_ARGUMENT, "ref / eval / out_gamma / dims / spacing_mm is NULL");
    int rc = check_criteria(DD, mode, low_dose_cutoff);
    if (rc) return rc;
    Resolved r;
    rc = resolve_opts(opts, r);
    if (rc) return rc;
    r.profile = 0;
    if (r.stats.hist || r.stats.summary)               // one pair of buffers cannot serve n cases
        return fail(GAMMA_ERR_INVALID_ARGUMENT, "gamma_eval_batch cannot honour opts.stats_*: use gamma_eval_ex per case or gamma_stats");
    // every case is checked before anything is enqueued: nothing is launched on an argument error
    for (int i = 0; i < n_cases; ++i) {
        if (!ref[i] || !eval[i] || !out_gamma[i]) return fail(GAMMA_ERR_INVALID_ARGUMENT, "ref[i] / eval[i] / out_gamma[i] is NULL");
        GridP g;
        rc = make_grid(dims + 3 * i, spacing_mm + 3 * i, DTA_mm, g);
        if (rc) return rc;
    }
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    std::lock_guard<std::mutex> lock(g_mu);
    cudaStreamCaptureStatus capStatus = cudaStreamCaptureStatusNone;
    CU_TRY(cudaStreamIsCapturing(st, &capStatus));
    if (capStatus != cudaStreamCaptureStatusNone)
        return fail(GAMMA_ERR_INVALID_ARGUMENT, "gamma_eval_batch cannot be captured into a CUDA graph; capture gamma_eval calls");
    // The cases run like back-to-back calls: round-robin over the library's lane streams, the first one after what is
    // already on `stream`, `stream` continues after the last; hazards between the cases' buffers are checked.
    for (int i = 0; i < n_cases; ++i) {
        GridP g;
        make_grid(dims + 3 * i, spacing_mm + 3 * i, DTA_mm, g);
        rc = enqueue_on_lane(ref[i], eval[i], g, DD, mode, low_dose_cutoff, r, out_gamma[i], st, i == 0);
        if (rc) return rc;
    }
    CU_TRY(cudaGetLastError());
    return GAMMA_OK;
}

int gamma_eval_general(const float* ref, const int ref_dims[3], const float ref_spacing_mm[3], const float ref_origin_mm[3],
                       const float* eval, const int eval_dims[3], const float eval_spacing_mm[3],
                       const float eval_origin_mm[3], float DD, float DTA_mm, int mode, float low_dose_cutoff,
                       const gamma_opts* opts, float* out_gamma, float* out_closest, void* stream)
{
    g_err.clear();
    if (!ref || !eval || !out_gamma) return fail(GAMMA_ERR_INVALID_ARGUMENT, "ref / eval / out_gamma is NULL");
    if (!ref_dims || !ref_spacing_mm || !ref_origin_mm || !eval_origin_mm)
        return fail(GAMMA_ERR_INVALID_ARGUMENT, "a geometry argument is NULL");
    GridP g;
    int rc = make_grid(eval_dims, eval_spacing_mm, DTA_mm, g);
    if (rc) return rc;
    if (!g.all_active) return fail(GAMMA_ERR_INVALID_ARGUMENT, "gamma_eval_general needs every evaluation axis >= 2 voxels");
    rc = check_criteria(DD, mode, low_dose_cutoff);
    if (rc) return rc;
    Resolved r;
    rc = resolve_opts(opts, r);
    if (rc) return rc;
    if (r.stats.hist || r.stats.summary)
        return fail(GAMMA_ERR_INVALID_ARGUMENT, "gamma_eval_general cannot honour opts.stats_*: run gamma_stats on out_gamma");
    GeneralP gp;
    std::memset(&gp, 0, sizeof gp);
    long long Nr = 1;
    for (int a = 0; a < 3; ++a) {
        if (ref_dims[a] < 1) return fail(GAMMA_ERR_INVALID_ARGUMENT, "ref_dims must be >= 1");
        if (!(ref_spacing_mm[a] > 0.0f) || !std::isfinite(ref_spacing_mm[a]))
            return fail(GAMMA_ERR_INVALID_ARGUMENT, "ref_spacing_mm must be > 0");
        if (!std::isfinite(ref_origin_mm[a]) || !std::isfinite(eval_origin_mm[a]))
            return fail(GAMMA_ERR_INVALID_ARGUMENT, "origins must be finite");
        Nr *= ref_dims[a];
        if (Nr >= (1ll << 31)) return fail(GAMMA_ERR_INVALID_ARGUMENT, "reference voxels must be < 2^31");
        gp.rn[a] = ref_dims[a];
        gp.off[a] = ((double)ref_origin_mm[a] - (double)eval_origin_mm[a]) / (double)eval_spacing_mm[a];
        gp.scale[a] = (double)ref_spacing_mm[a] / (double)eval_spacing_mm[a];
        gp.eorg[a] = eval_origin_mm[a];
        gp.esp[a] = eval_spacing_mm[a];
    }
    {
        const unsigned dv[2] = {(unsigned)ref_dims[0], (unsigned)ref_dims[0] * (unsigned)ref_dims[1]};
        for (int k = 0; k < 2; ++k) {
            unsigned l = 0;
            while ((1ull << l) < dv[k]) ++l;
            gp.rDivMul[k] = (unsigned)((1ull << (31 + l)) / dv[k] + 1ull);
            gp.rDivSh[k] = 31 + l;
        }
    }
    GridP gr;                                   // the reference grid as k_classify sees it: a run of Nr voxels
    std::memset(&gr, 0, sizeof gr);
    gr.n[0] = ref_dims[0]; gr.n[1] = ref_dims[1]; gr.n[2] = ref_dims[2];
    gr.stride[0] = 1; gr.stride[1] = ref_dims[0]; gr.stride[2] = ref_dims[0] * ref_dims[1];
    gr.N = (int)Nr;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    std::lock_guard<std::mutex> lock(g_mu);
    end_b2b_sequence();
    cudaStreamCaptureStatus capStatus = cudaStreamCaptureStatusNone;
    CU_TRY(cudaStreamIsCapturing(st, &capStatus));
    if (capStatus != cudaStreamCaptureStatusNone)
        return fail(GAMMA_ERR_INVALID_ARGUMENT, "gamma_eval_general cannot be captured into a CUDA graph");
    rc = ensure_device();
    if (rc) return rc;
    rc = order_after_previous(st);
    if (rc) return rc;
    rc = ensure_ctl(st);
    if (rc) return rc;
    g_ws.ctlClean = false;
    rc = prepare_workspace(g, r, Nr);
    if (rc) return rc;
    Ctl* base = static_cast<Ctl*>(g_ws.ctl.p);
    Ctl* ctl = base + g_ws.slot;
    Ctl* next = base + (g_ws.slot + 1) % CTL_ROT;
    EvalP e;
    e.DD = DD; e.cutoff = low_dose_cutoff; e.norm_dose = r.normDose; e.mode = mode; e.algo = 0; e.call = g_callNo;
    const int sm = g_ws.numSM;
    const bool pdl = g_ws.pdl != 0;
    StatsP noStats;
    noStats.hist = nullptr; noStats.summary = nullptr; noStats.nbins = 0; noStats.binScale = 0.0f;
    {                                                                    // a0 on the reference grid
        long long blocks = (Nr + 1023) / 1024;
        int grid = (int)(blocks < 1 ? 1 : (blocks > sm * 4 ? sm * 4 : blocks));
        CU_TRY(launch_ex(k_norm, grid, NORM_THREADS, 0, st, pdl, false, ref, ref, (int)Nr, mode, ctl, next, 1, e.call, noStats, 0));
    }
    {                                                                    // a1 on the reference grid
        long long chunks = (Nr + PREP_CHUNK - 1) / PREP_CHUNK;
        int grid = (int)(chunks > sm * 8 ? sm * 8 : chunks);
        CU_TRY(launch_ex(k_classify, grid, PREP_THREADS, 0, st, pdl, false, ref, out_gamma, gr, e, ctl,
                         static_cast<unsigned*>(g_ws.evalIdx.p), noStats, static_cast<Ctl*>(nullptr), 0));
    }
    // a3 on the evaluation grid: the same data-independent prefix table as gamma_eval (table_cap cells), here by the
    // stand-alone builder; beyond it the search enumerates
    const bool embed = r.tableCap <= TAB_EMBED_MAX_CELLS;
    int4* tab = static_cast<int4*>(g_ws.table.p) + (embed ? (size_t)g_ws.slot * TAB_EMBED_MAX_CELLS : (size_t)CTL_SLOTS * TAB_EMBED_MAX_CELLS);
    {
        float lo = 0.0f, hi = grid_diagonal(g);
        int bx, by, bz;
        if (table_box_cells(g, hi, bx, by, bz) <= r.tableCap) lo = hi;
        else
            for (int it = 0; it < 48; ++it) {
                const float mid = 0.5f * (lo + hi);
                if (table_box_cells(g, mid, bx, by, bz) <= r.tableCap) lo = mid; else hi = mid;
            }
        k_offset_table<<<TAB_BLOCKS, TAB_THREADS, TAB_DYN_SMEM, st>>>(g, e, ctl, lo, r.tableCap, tab, static_cast<unsigned*>(g_ws.tmpL.p),
                                                                      static_cast<unsigned*>(g_ws.tmpIdx.p), 1);
    }
    if (out_closest) CU_TRY(cudaMemsetAsync(out_closest, 0xff, (size_t)Nr * 16, st));   // NaN where nothing is evaluated
    {
        long long units = (Nr + 3) / 4, blocks = (units + GENERAL_THREADS / 32 - 1) / (GENERAL_THREADS / 32);
        if (g_ws.occGeneral == 0) {
            int occ = 0;
            CU_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_general_search, GENERAL_THREADS, 0));
            g_ws.occGeneral = occ > 0 ? occ : 1;
        }
        const long long resident = (long long)sm * g_ws.occGeneral;
        const int grid = (int)(blocks > resident ? resident : (blocks < 1 ? 1 : blocks));
        CU_TRY(launch_ex(k_general_search, grid, GENERAL_THREADS, 0, st, false, false, ref, eval, out_gamma,
                         reinterpret_cast<float4*>(out_closest), g, gp, e, ctl, static_cast<const unsigned*>(g_ws.evalIdx.p),
                         static_cast<const int4*>(tab)));
    }
    g_ws.launches += 4;
    CU_TRY(cudaGetLastError());
    rc = mark_done(st);
    if (rc) return rc;
    g_ws.lastSpans = CallSpans();
    g_ws.lastCtl = ctl;
    g_ws.lastClasses = 0;
    g_ws.slot = (g_ws.slot + 1) % CTL_ROT;
    ++g_ws.calls;
    ++g_callNo;
    g_ws.ctlClean = true;
    g_ws.lastStream = st; g_ws.lastN = Nr; g_ws.haveLast = true; g_ws.haveStages = false;
    g_lastWs = g_cur;
    return GAMMA_OK;
}

int gamma_eval_host(const float* ref_host, const float* eval_host, const int dims[3], const float spacing_mm[3],
                    float DD, float DTA_mm, int mode, float low_dose_cutoff, const gamma_opts* opts,
                    float* out_gamma_host, void* stream)
{
    g_err.clear();
    if (!ref_host || !eval_host || !out_gamma_host)
        return fail(GAMMA_ERR_INVALID_ARGUMENT, "ref_host / eval_host / out_gamma_host is NULL");
    GridP g;
    int rc = make_grid(dims, spacing_mm, DTA_mm, g);
    if (rc) return rc;
    rc = check_criteria(DD, mode, low_dose_cutoff);
    if (rc) return rc;
    Resolved r;
    rc = resolve_opts(opts, r);
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    std::lock_guard<std::mutex> lock(g_mu);
    end_b2b_sequence();
    const size_t bytes = (size_t)g.N * 4;
    CU_TRY(g_ws.hRef.need(bytes)); CU_TRY(g_ws.hEval.need(bytes)); CU_TRY(g_ws.hOut.need(bytes));
    rc = order_after_previous(st);
    if (rc) return rc;
    CU_TRY(cudaMemcpyAsync(g_ws.hRef.p, ref_host, bytes, cudaMemcpyHostToDevice, st));     // A2 step 1
    CU_TRY(cudaMemcpyAsync(g_ws.hEval.p, eval_host, bytes, cudaMemcpyHostToDevice, st));
    rc = enqueue_pipeline(static_cast<const float*>(g_ws.hRef.p), static_cast<const float*>(g_ws.hEval.p), g, DD, mode,
                          low_dose_cutoff, r, static_cast<float*>(g_ws.hOut.p), st, false);
    if (rc) return rc;
    CU_TRY(cudaMemcpyAsync(out_gamma_host, g_ws.hOut.p, bytes, cudaMemcpyDeviceToHost, st)); // A2 step 8
    rc = mark_done(st);
    if (rc) return rc;
    CU_TRY(cudaStreamSynchronize(st));
    return GAMMA_OK;
}

int gamma_eval_host_batch(int n_cases, const float* const* ref_host, const float* const* eval_host, const int* dims,
                          const float* spacing_mm, float DD, float DTA_mm, int mode, float low_dose_cutoff,
                          const gamma_opts* opts, float* const* out_gamma_host, void* stream)
{
    g_err.clear();
    if (n_cases < 0) return fail(GAMMA_ERR_INVALID_ARGUMENT, "n_cases must be >= 0");
    if (n_cases == 0) return GAMMA_OK;
    if (!ref_host || !eval_host || !out_gamma_host || !dims || !spacing_mm)
        return fail(GAMMA_ERR_INVALID_ARGUMENT, "ref_host / eval_host / out_gamma_host / dims / spacing_mm is NULL");
    int rc = check_criteria(DD, mode, low_dose_cutoff);
    if (rc) return rc;
    Resolved r;
    rc = resolve_opts(opts, r);
    if (rc) return rc;
    r.profile = 0; r.graph = 0;
    if (r.stats.hist || r.stats.summary)
        return fail(GAMMA_ERR_INVALID_ARGUMENT, "gamma_eval_host_batch cannot honour opts.stats_*: use gamma_eval_host per case or gamma_stats");
    long long maxN = 0;
    for (int i = 0; i < n_cases; ++i) {                  // every case is checked before anything is enqueued
        if (!ref_host[i] || !eval_host[i] || !out_gamma_host[i])
            return fail(GAMMA_ERR_INVALID_ARGUMENT, "ref_host[i] / eval_host[i] / out_gamma_host[i] is NULL");
        GridP g;
        rc = make_grid(dims + 3 * i, spacing_mm + 3 * i, DTA_mm, g);
        if (rc) return rc;
        if (g.N > maxN) maxN = g.N;
    }
    cudaStream_t user = static_cast<cudaStream_t>(stream);
    std::lock_guard<std::mutex> lock(g_mu);
    end_b2b_sequence();
    cudaStreamCaptureStatus capStatus = cudaStreamCaptureStatusNone;
    CU_TRY(cudaStreamIsCapturing(user, &capStatus));
    if (capStatus != cudaStreamCaptureStatusNone)
        return fail(GAMMA_ERR_INVALID_ARGUMENT, "gamma_eval_host_batch synchronises and cannot be captured into a CUDA graph");
    rc = lanes_init();
    if (rc) return rc;
    HostBatchState& H = g_hb;
    if (!H.ready) {
        CU_TRY(cudaStreamCreateWithFlags(&H.h2d, cudaStreamNonBlocking));
        CU_TRY(cudaStreamCreateWithFlags(&H.d2h, cudaStreamNonBlocking));
        CU_TRY(cudaEventCreateWithFlags(&H.start, cudaEventDisableTiming));
        for (int k = 0; k < HB_DEPTH; ++k) {
            CU_TRY(cudaEventCreateWithFlags(&H.copied[k], cudaEventDisableTiming));
            CU_TRY(cudaEventCreateWithFlags(&H.computed[k], cudaEventDisableTiming));
            CU_TRY(cudaEventCreateWithFlags(&H.freed[k], cudaEventDisableTiming));
        }
        H.ready = true;
    }
    const int depth = n_cases < HB_DEPTH ? n_cases : HB_DEPTH;
    for (int k = 0; k < depth; ++k) {
        CU_TRY(H.ref[k].need((size_t)maxN * 4)); CU_TRY(H.ev[k].need((size_t)maxN * 4)); CU_TRY(H.out[k].need((size_t)maxN * 4));
    }
    cudaStream_t comp = g_lanes.stream[0];
    CU_TRY(cudaEventRecord(H.start, user));              // everything starts after what is already on `stream`
    CU_TRY(cudaStreamWaitEvent(H.h2d, H.start, 0));
    g_lanes.laneDirty[0] = true;
    // A failure inside the loop must not return while copies that were already enqueued may still read or write the
    // caller's host buffers: note it, stop enqueuing, synchronise the three streams below, then report it.
    cudaError_t ce = cudaSuccess;
    const char* ceWhere = "";
#define HB_TRY(call) { ce = (call); if (ce != cudaSuccess) { ceWhere = #call; break; } }
    for (int i = 0; i < n_cases; ++i) {
        const int k = i % HB_DEPTH;
        GridP g;
        make_grid(dims + 3 * i, spacing_mm + 3 * i, DTA_mm, g);
        const size_t bytes = (size_t)g.N * 4;
        if (i >= HB_DEPTH) HB_TRY(cudaStreamWaitEvent(H.h2d, H.freed[k], 0));          // set k has been read back
        HB_TRY(cudaMemcpyAsync(H.ref[k].p, ref_host[i], bytes, cudaMemcpyHostToDevice, H.h2d));      // A2 step 1
        HB_TRY(cudaMemcpyAsync(H.ev[k].p, eval_host[i], bytes, cudaMemcpyHostToDevice, H.h2d));
        HB_TRY(cudaEventRecord(H.copied[k], H.h2d));
        HB_TRY(cudaStreamWaitEvent(comp, H.copied[k], 0));
        Workspace* keep = g_cur;
        g_cur = &g_pool[1];
        rc = enqueue_pipeline(static_cast<const float*>(H.ref[k].p), static_cast<const float*>(H.ev[k].p), g, DD, mode,
                              low_dose_cutoff, r, static_cast<float*>(H.out[k].p), comp, false);
        g_cur = keep;
        if (rc) break;
        HB_TRY(cudaEventRecord(H.computed[k], comp));
        HB_TRY(cudaStreamWaitEvent(H.d2h, H.computed[k], 0));
        HB_TRY(cudaMemcpyAsync(out_gamma_host[i], H.out[k].p, bytes, cudaMemcpyDeviceToHost, H.d2h));  // A2 step 8
        HB_TRY(cudaEventRecord(H.freed[k], H.d2h));
    }
#undef HB_TRY
    cudaError_t e1 = cudaStreamSynchronize(H.d2h), e2 = cudaStreamSynchronize(comp), e3 = cudaStreamSynchronize(H.h2d);
    if (rc) return rc;
    if (ce != cudaSuccess)
        return fail(ce == cudaErrorMemoryAllocation ? GAMMA_ERR_OUT_OF_MEMORY : GAMMA_ERR_CUDA,
                    std::string(ceWhere) + ": " + cudaGetErrorString(ce));
    CU_TRY(e1); CU_TRY(e2); CU_TRY(e3);
    return GAMMA_OK;
}

int gamma_stats(const float* gamma, long long n, int nbins, float hist_max, unsigned long long* hist_dev,
                gamma_summary* out_dev, void* stream)
{
    g_err.clear();
    if (n < 0 || n >= (1ll << 40)) return fail(GAMMA_ERR_INVALID_ARGUMENT, "n out of range");
    if ((!gamma && n > 0) || !hist_dev || !out_dev)
        return fail(GAMMA_ERR_INVALID_ARGUMENT, "gamma / hist_dev / out_dev is NULL");
    if (nbins < 1 || nbins > STATS_MAX_BINS) return fail(GAMMA_ERR_INVALID_ARGUMENT, "nbins must be in [1, 4096]");
    if (!(hist_max > 0.0f) || !std::isfinite(hist_max)) return fail(GAMMA_ERR_INVALID_ARGUMENT, "hist_max must be > 0");
    std::lock_guard<std::mutex> lock(g_mu);
    end_b2b_sequence();
    int rc = ensure_device();
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    k_stats_clear<<<(nbins + 255) / 256, 256, 0, st>>>(hist_dev, nbins, out_dev);
    if (n > 0) {
        long long blocks = (n + STATS_THREADS * 8 - 1) / (STATS_THREADS * 8);
        int grid = (int)(blocks > g_ws.numSM * 4 ? g_ws.numSM * 4 : blocks);
        const size_t smem = (size_t)nbins * (nbins <= STATS_WARP_BINS ? STATS_WARPS : 1) * sizeof(unsigned);
        CU_TRY(launch_ex(k_stats, grid, STATS_THREADS, smem, st, true, false, gamma, n, nbins, (float)nbins / hist_max,
                         hist_dev, out_dev));
        ++g_ws.launches;
    }
    ++g_ws.launches;
    CU_TRY(cudaGetLastError());
    return GAMMA_OK;
}

__global__ void k_set_u32(unsigned* p, unsigned v) { *p = v; }

int gamma_sort_pairs(unsigned int* keys, unsigned int* vals, long long n, int begin_bit, int end_bit, void* stream)
{
    g_err.clear();
    if (n < 0 || n >= (1ll << 31)) return fail(GAMMA_ERR_INVALID_ARGUMENT, "n must be in [0, 2^31)");
    if (n > 0 && (!keys || !vals)) return fail(GAMMA_ERR_INVALID_ARGUMENT, "keys / vals is NULL");
    if (begin_bit < 0 || end_bit > 32 || begin_bit >= end_bit || (begin_bit & 7) || (end_bit & 7))
        return fail(GAMMA_ERR_INVALID_ARGUMENT, "need 0 <= begin_bit < end_bit <= 32, multiples of 8");
    if (n == 0) return GAMMA_OK;
    std::lock_guard<std::mutex> lock(g_mu);
    end_b2b_sequence();
    int rc = ensure_device();
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const long long maxTiles = (n + SORT_TILE - 1) / SORT_TILE;
    rc = ensure_ctl(st);
    if (rc) return rc;
    CU_TRY(g_ws.sortK.need(n * 4)); CU_TRY(g_ws.sortV.need(n * 4));
    CU_TRY(g_ws.tileHist.need((size_t)(maxTiles + 1) * SORT_RADIX * 4));             // + the 256 digit totals
    rc = order_after_previous(st);
    if (rc) return rc;
    Ctl* ctl = static_cast<Ctl*>(g_ws.ctl.p) + CTL_STANDALONE;
    k_set_u32<<<1, 1, 0, st>>>(&ctl->sortN, (unsigned)n);
    unsigned *k1 = static_cast<unsigned*>(g_ws.sortK.p), *v1 = static_cast<unsigned*>(g_ws.sortV.p);
    int where = radix_sort_enqueue(keys, vals, k1, v1, &ctl->sortN, n, begin_bit, end_bit,
                                   static_cast<unsigned*>(g_ws.tileHist.p), st);
    g_ws.launches += 1 + 3 * ((end_bit - begin_bit) / 8);
    if (where) {
        CU_TRY(cudaMemcpyAsync(keys, k1, n * 4, cudaMemcpyDeviceToDevice, st));
        CU_TRY(cudaMemcpyAsync(vals, v1, n * 4, cudaMemcpyDeviceToDevice, st));
    }
    CU_TRY(cudaGetLastError());
    return mark_done(st);
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------------
// gamma_sort_pairs_noalloc: the same radix sort for callers that must not allocate device memory.
//
// gamma_sort_pairs takes its ping-pong buffers, tile histograms and element counter from the library's grow-only
// workspace, i.e. from cudaMalloc on first use and whenever n grows.  That is not an option for a caller that
//   * runs while some thread of the process is capturing a stream in the global capture mode (cudaMalloc is refused
//     there, and a refused call breaks the capture),
//   * sits in a latency-critical loop (cudaMalloc / cudaFree synchronise the device and cost 0.1 - 1 ms), or
//   * lives in a process whose device memory is handed out by one pool (the PyTorch caching allocator, a treatment
//     planning system's arena) that has reserved all there is, so that a side allocation fails or fragments it.
// For them the scratch lives in the library image itself: the file-scope array below, SORT_NOALLOC_WORDS * 4 bytes
// (about 8.3 MB) of every GPU on which the library's module is loaded, held until the process exits.  The array is one
// object per device.  Its name in HOST code is a stand-in, not an address a kernel could use; the address on the current
// device comes from cudaGetSymbolAddress, asked once per device with that device current (noalloc_scratch()).
//
// Layout, in 32-bit words: [0, MAX) second key buffer | [MAX, 2 MAX) second value buffer | tile histograms
// (256 x tiles, + 256 digit totals) | the element counter the kernels read n from.
// Nothing in it has to start at zero: k_radix_hist writes every histogram word k_radix_scan and k_radix_scatter read,
// k_radix_scan writes the digit totals, k_set_u32 the counter, and a pass overwrites the part of the ping-pong buffers the
// next one reads.  What a call leaves behind is therefore harmless to the next call -- as long as the two do not overlap
// on the device, see the header.
constexpr long long SORT_NOALLOC_MAX = GAMMA_SORT_NOALLOC_MAX_PAIRS;
constexpr size_t SORT_NOALLOC_TILES = (size_t)((SORT_NOALLOC_MAX + SORT_TILE - 1) / SORT_TILE);
constexpr size_t SORT_NOALLOC_VALS = (size_t)SORT_NOALLOC_MAX;                  // word offsets, multiples of 64 (256 B)
constexpr size_t SORT_NOALLOC_HIST = 2 * (size_t)SORT_NOALLOC_MAX;
constexpr size_t SORT_NOALLOC_COUNT = SORT_NOALLOC_HIST + (SORT_NOALLOC_TILES + 1) * SORT_RADIX;
constexpr size_t SORT_NOALLOC_WORDS = SORT_NOALLOC_COUNT + 64;
static_assert(SORT_NOALLOC_MAX % 64 == 0, "keeps the parts of the scratch array 256-byte aligned");
static __device__ __align__(256) unsigned g_sortNoallocScratch[SORT_NOALLOC_WORDS];

namespace {
constexpr int NOALLOC_MAX_DEVICES = 64;
unsigned* g_sortNoallocPtr[NOALLOC_MAX_DEVICES] = {};   // device address of g_sortNoallocScratch, per device ordinal

// Device address of the scratch array on the CURRENT device (looked up on the first call per device; g_mu held).
int noalloc_scratch(unsigned** out)
{
    int dev = -1;
    CU_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return fail(GAMMA_ERR_INVALID_ARGUMENT, "device ordinal above 63");
    if (!g_sortNoallocPtr[dev]) {
        unsigned* p = nullptr;
        CU_TRY(cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_sortNoallocScratch));
        if (!p) return fail(GAMMA_ERR_CUDA, "cudaGetSymbolAddress returned a null address for the sort scratch");
        g_sortNoallocPtr[dev] = p;
    }
    *out = g_sortNoallocPtr[dev];
    return GAMMA_OK;
}
}  // namespace

extern "C" {

int gamma_sort_pairs_noalloc(unsigned int* keys, unsigned int* vals, long long n, int begin_bit, int end_bit,
                             void* stream)
{
    g_err.clear();
    if (n < 0) return fail(GAMMA_ERR_INVALID_ARGUMENT, "n must be >= 0");
    if (n > SORT_NOALLOC_MAX)
        return fail(GAMMA_ERR_INVALID_ARGUMENT,
                    "gamma_sort_pairs_noalloc: n = " + std::to_string(n) + " exceeds GAMMA_SORT_NOALLOC_MAX_PAIRS = " +
                        std::to_string(SORT_NOALLOC_MAX) + " (the built-in scratch); use gamma_sort_pairs");
    if (n > 0 && (!keys || !vals)) return fail(GAMMA_ERR_INVALID_ARGUMENT, "keys / vals is NULL");
    if (begin_bit < 0 || end_bit > 32 || begin_bit >= end_bit || (begin_bit & 7) || (end_bit & 7))
        return fail(GAMMA_ERR_INVALID_ARGUMENT, "need 0 <= begin_bit < end_bit <= 32, multiples of 8");
    if (n == 0) return GAMMA_OK;
    std::lock_guard<std::mutex> lock(g_mu);
    end_b2b_sequence();                    // a host flag: a sort on `stream` ends a sequence of back-to-back gamma calls
    unsigned* scratch = nullptr;
    int rc = noalloc_scratch(&scratch);
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    unsigned *k1 = scratch, *v1 = scratch + SORT_NOALLOC_VALS, *tileHist = scratch + SORT_NOALLOC_HIST;
    unsigned* count = scratch + SORT_NOALLOC_COUNT;
    k_set_u32<<<1, 1, 0, st>>>(count, (unsigned)n);
    // tileHist is laid out for ceil(n / SORT_TILE) tiles by the kernels and by radix_sort_enqueue alike (<= SORT_NOALLOC_TILES)
    int where = radix_sort_enqueue(keys, vals, k1, v1, count, n, begin_bit, end_bit, tileHist, st);
    g_pool[0].launches += 1 + 3 * ((end_bit - begin_bit) / 8);
    if (where) {    // an odd number of passes ends in the scratch: bring the result home (device-to-device, no staging)
        CU_TRY(cudaMemcpyAsync(keys, k1, (size_t)n * 4, cudaMemcpyDeviceToDevice, st));
        CU_TRY(cudaMemcpyAsync(vals, v1, (size_t)n * 4, cudaMemcpyDeviceToDevice, st));
    }
    CU_TRY(cudaGetLastError());
    return GAMMA_OK;
}

__global__ void k_table_export(const Ctl* __restrict__ ctl, const int4* __restrict__ table, long long maxEntries,
                               int* __restrict__ outEntries, int* __restrict__ outCount)
{
    const unsigned T = ctl->tableCount;
    const unsigned lim = (unsigned)(T < maxEntries ? T : maxEntries);
    for (unsigned i = blockIdx.x * blockDim.x + threadIdx.x; i < lim; i += gridDim.x * blockDim.x) {
        const int4 t = table[i];
        outEntries[4 * i + 0] = t.x; outEntries[4 * i + 1] = t.y; outEntries[4 * i + 2] = t.z; outEntries[4 * i + 3] = t.w;
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        outCount[0] = (int)lim;
        outCount[1] = (int)ctl->tableTrunc;
        outCount[2] = __float_as_int(ctl->Rtab2);
    }
}

int gamma_offset_table(const int dims[3], const float spacing_mm[3], float DTA_mm, float radius, long long max_entries,
                       int* out_entries, int* out_count, void* stream)
{
    g_err.clear();
    if (!out_entries || !out_count) return fail(GAMMA_ERR_INVALID_ARGUMENT, "out_entries / out_count is NULL");
    if (!(radius >= 0.0f) || !std::isfinite(radius)) return fail(GAMMA_ERR_INVALID_ARGUMENT, "radius must be >= 0");
    if (max_entries < 1 || max_entries > (1ll << 26)) return fail(GAMMA_ERR_INVALID_ARGUMENT, "max_entries must be in [1, 2^26]");
    GridP g;
    int rc = make_grid(dims, spacing_mm, DTA_mm, g);
    if (rc) return rc;
    std::lock_guard<std::mutex> lock(g_mu);
    end_b2b_sequence();
    rc = ensure_device();
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    rc = ensure_ctl(st);
    if (rc) return rc;
    CU_TRY(g_ws.table.need((size_t)max_entries * 16));
    CU_TRY(g_ws.tmpL.need((size_t)max_entries * 4)); CU_TRY(g_ws.tmpIdx.need((size_t)max_entries * 4));
    CU_TRY(cudaFuncSetAttribute(k_offset_table, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TAB_DYN_SMEM));
    rc = order_after_previous(st);
    if (rc) return rc;
    Ctl* ctl = static_cast<Ctl*>(g_ws.ctl.p) + CTL_STANDALONE;
    EvalP e;
    e.DD = 1.0f; e.cutoff = 0.0f; e.norm_dose = 1.0f; e.mode = 0; e.algo = 0; e.call = 0;
    k_offset_table<<<TAB_BLOCKS, TAB_THREADS, TAB_DYN_SMEM, st>>>(
        g, e, ctl, radius, max_entries, static_cast<int4*>(g_ws.table.p), static_cast<unsigned*>(g_ws.tmpL.p),
        static_cast<unsigned*>(g_ws.tmpIdx.p), 0);
    k_table_export<<<64, 256, 0, st>>>(ctl, static_cast<const int4*>(g_ws.table.p), max_entries, out_entries, out_count);
    g_ws.launches += 2;
    CU_TRY(cudaGetLastError());
    g_ws.haveLast = false;
    return mark_done(st);
}

int gamma_get_counters(gamma_counters* out_host)
{
    g_err.clear();
    if (!out_host) return fail(GAMMA_ERR_INVALID_ARGUMENT, "out_host is NULL");
    std::lock_guard<std::mutex> lock(g_mu);
    const Workspace& w = *g_lastWs;                  // the workspace the last gamma_eval* call ran on
    if (!w.haveLast || !w.ctl.p) return fail(GAMMA_ERR_INVALID_ARGUMENT, "no gamma_eval call to report on");
    if (w.lastStream) CU_TRY(cudaStreamSynchronize(w.lastStream));
    else CU_TRY(cudaDeviceSynchronize());            // last call was captured by the caller: no stream to wait on
    Ctl c;
    CU_TRY(cudaMemcpy(&c, w.lastCtl, sizeof c, cudaMemcpyDeviceToHost));
    std::memset(out_host, 0, sizeof *out_host);
    out_host->n_voxels = w.lastN;
    out_host->n_evaluated = c.nEval;
    out_host->n_table_search = (long long)c.nSearch + (long long)c.nDeep;
    out_host->table_entries = c.tableCount;
    out_host->vertex_visits = (long long)c.visits;
    union { unsigned u; float f; } cv;
    cv.u = c.maxKeyBits;
    out_host->max_key = cv.f;
    out_host->norm_dose = w.lastNormDose > 0.0f ? w.lastNormDose : ordered_to_float(c.normOrd);
    out_host->table_truncated = (int)c.tableTrunc;
    out_host->n_ring_search = w.lastClasses ? (int)c.nSearch : 0;
    out_host->pipelined = (&w != &g_pool[0] && &w != &g_pool[WS_CAPTURE]) ? 1 : 0;
    out_host->calls_pipelined = (long long)g_lanes.next;
    return GAMMA_OK;
}

int gamma_get_stage_times(gamma_stage_times* out_host)
{
    g_err.clear();
    if (!out_host) return fail(GAMMA_ERR_INVALID_ARGUMENT, "out_host is NULL");
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_ws.haveStages) return fail(GAMMA_ERR_INVALID_ARGUMENT, "last gamma_eval call did not set opts.profile_stages");
    CU_TRY(cudaEventSynchronize(g_ws.stage[4]));
    if (g_ws.stageTable) CU_TRY(cudaEventSynchronize(g_ws.stage[6]));
    CU_TRY(cudaEventElapsedTime(&out_host->prep_ms, g_ws.stage[0], g_ws.stage[1]));
    CU_TRY(cudaEventElapsedTime(&out_host->star_ms, g_ws.stage[1], g_ws.stage[2]));
    out_host->sort_ms = 0.0f;
    if (g_ws.stageSort) CU_TRY(cudaEventElapsedTime(&out_host->sort_ms, g_ws.stage[2], g_ws.stage[3]));
    CU_TRY(cudaEventElapsedTime(&out_host->search_ms, g_ws.stage[g_ws.stageSort ? 3 : 2], g_ws.stage[4]));
    out_host->table_ms = 0.0f;
    if (g_ws.stageTable) CU_TRY(cudaEventElapsedTime(&out_host->table_ms, g_ws.stage[5], g_ws.stage[6]));
    CU_TRY(cudaEventElapsedTime(&out_host->total_ms, g_ws.stage[0], g_ws.stage[4]));
    return GAMMA_OK;
}

long long gamma_launch_count(void)
{
    std::lock_guard<std::mutex> lock(g_mu);
    long long n = 0;
    for (const Workspace& w : g_pool) n += w.launches;
    return n;
}

// ---- device timeline (GAMMA_TRACE builds; common.cuh)
#ifdef GAMMA_TRACE
namespace { TraceRec* g_traceDev = nullptr; TraceWarp* g_traceWarpsDev = nullptr; }
#endif
int gamma_trace_reset(void)
{
    g_err.clear();
#ifdef GAMMA_TRACE
    std::lock_guard<std::mutex> lock(g_mu);
    CU_TRY(cudaDeviceSynchronize());
    const size_t n = (size_t)TRACE_CALLS * TRACE_KERNELS;
    if (!g_traceDev) CU_TRY(cudaMalloc(&g_traceDev, n * sizeof(TraceRec)));
    static TraceRec init[TRACE_CALLS * TRACE_KERNELS];
    for (size_t i = 0; i < n; ++i) { init[i].first = ~0ull; init[i].waited = 0; init[i].last = 0; init[i].pad_ = 0; }
    CU_TRY(cudaMemcpy(g_traceDev, init, n * sizeof(TraceRec), cudaMemcpyHostToDevice));
    CU_TRY(cudaMemcpyToSymbol(g_trace_buf, &g_traceDev, sizeof g_traceDev));
    if (!g_traceWarpsDev) CU_TRY(cudaMalloc(&g_traceWarpsDev, (size_t)TRACE_WARPS * sizeof(TraceWarp)));
    CU_TRY(cudaMemset(g_traceWarpsDev, 0, (size_t)TRACE_WARPS * sizeof(TraceWarp)));
    CU_TRY(cudaMemcpyToSymbol(g_trace_warps, &g_traceWarpsDev, sizeof g_traceWarpsDev));
    return GAMMA_OK;
#else
    return fail(GAMMA_ERR_INVALID_ARGUMENT, "libgamma_b200 was built without -DGAMMA_TRACE");
#endif
}

int gamma_trace_read(unsigned long long* out_host, long long* next_call)
{
    g_err.clear();
#ifdef GAMMA_TRACE
    if (!out_host || !next_call) return fail(GAMMA_ERR_INVALID_ARGUMENT, "out_host / next_call is NULL");
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_traceDev) return fail(GAMMA_ERR_INVALID_ARGUMENT, "gamma_trace_reset has not been called");
    CU_TRY(cudaDeviceSynchronize());
    CU_TRY(cudaMemcpy(out_host, g_traceDev, (size_t)TRACE_CALLS * TRACE_KERNELS * sizeof(TraceRec), cudaMemcpyDeviceToHost));
    *next_call = (long long)g_callNo;
    return GAMMA_OK;
#else
    (void)out_host; (void)next_call;
    return fail(GAMMA_ERR_INVALID_ARGUMENT, "libgamma_b200 was built without -DGAMMA_TRACE");
#endif
}

int gamma_trace_read_warps(unsigned long long* out_host, int max_warps)
{
    g_err.clear();
#ifdef GAMMA_TRACE
    if (!out_host || max_warps < 1) return fail(GAMMA_ERR_INVALID_ARGUMENT, "out_host is NULL or max_warps < 1");
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_traceWarpsDev) return fail(GAMMA_ERR_INVALID_ARGUMENT, "gamma_trace_reset has not been called");
    CU_TRY(cudaDeviceSynchronize());
    const int n = max_warps < TRACE_WARPS ? max_warps : TRACE_WARPS;
    CU_TRY(cudaMemcpy(out_host, g_traceWarpsDev, (size_t)n * sizeof(TraceWarp), cudaMemcpyDeviceToHost));
    return GAMMA_OK;
#else
    (void)out_host; (void)max_warps;
    return fail(GAMMA_ERR_INVALID_ARGUMENT, "libgamma_b200 was built without -DGAMMA_TRACE");
#endif
}

long long gamma_workspace_bytes(void)
{
    std::lock_guard<std::mutex> lock(g_mu);
    size_t n = 0;
    for (const Workspace& w : g_pool) n += w.bytes();
    for (int k = 0; k < HB_DEPTH; ++k) n += g_hb.ref[k].cap + g_hb.ev[k].cap + g_hb.out[k].cap;   // gamma_eval_host_batch
    return (long long)n;
}

int gamma_fp32_probe(int repeats, double* out_tflops, void* stream)
{
    g_err.clear();
    if (!out_tflops || repeats < 1 || repeats > 1000) return fail(GAMMA_ERR_INVALID_ARGUMENT, "bad probe arguments");
    std::lock_guard<std::mutex> lock(g_mu);
    int rc = ensure_device();
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    rc = ensure_ctl(st);
    if (rc) return rc;
    cudaEvent_t a, b;
    CU_TRY(cudaEventCreate(&a)); CU_TRY(cudaEventCreate(&b));
    const int grid = g_ws.numSM * 8 * 4, threads = 256;
    double best = 0.0;
    for (int r = 0; r < repeats + 1; ++r) {
        CU_TRY(cudaEventRecord(a, st));
        k_fp32_probe<<<grid, threads, 0, st>>>(reinterpret_cast<float*>(static_cast<Ctl*>(g_ws.ctl.p) + CTL_STANDALONE) + 15, 0.999f, 1e-3f);
        ++g_ws.launches;
        CU_TRY(cudaEventRecord(b, st));
        CU_TRY(cudaEventSynchronize(b));
        float ms = 0.0f;
        CU_TRY(cudaEventElapsedTime(&ms, a, b));
        const double flops = 2.0 * (double)grid * threads * PROBE_ITERS * PROBE_CHAINS;
        if (r > 0 && ms > 0.0f) best = std::max(best, flops / (ms * 1e-3) / 1e12);
    }
    cudaEventDestroy(a); cudaEventDestroy(b);
    CU_TRY(cudaGetLastError());
    *out_tflops = best;
    return GAMMA_OK;
}

void gamma_release(void)
{
    std::lock_guard<std::mutex> lock(g_mu);
    cudaDeviceSynchronize();
#ifdef GAMMA_HOSTPROF
    for (int k = 0; k < 10; ++k)
        if (g_hp.n[k])
            std::fprintf(stderr, "[gamma hostprof] %-22s %10lld x %8.3f us = %10.1f us\n", HP_NAMES[k], g_hp.n[k],
                         g_hp.us[k] / (double)g_hp.n[k], g_hp.us[k]);
    g_hp = HostProf();
#endif
    for (Workspace& w : g_pool) w.releaseAll();
    for (int l = 0; l < LANES; ++l)
        if (g_lanes.stream[l]) { cudaStreamDestroy(g_lanes.stream[l]); g_lanes.stream[l] = nullptr; }
    for (int w = 0; w < B2B_WINDOW; ++w)
        if (g_lanes.done[w]) { cudaEventDestroy(g_lanes.done[w]); g_lanes.done[w] = nullptr; }
    if (g_lanes.fork) { cudaEventDestroy(g_lanes.fork); g_lanes.fork = nullptr; }
    if (g_lanes.joined) { cudaEventDestroy(g_lanes.joined); g_lanes.joined = nullptr; }
    if (g_lanes.join) { cudaStreamDestroy(g_lanes.join); g_lanes.join = nullptr; }
    g_lanes = LaneState();
    g_hb.release();
    g_lastWs = &g_pool[0];
}

void gamma_abi_sizes(int out_host[4])
{
    if (!out_host) return;
    out_host[0] = (int)sizeof(gamma_opts); out_host[1] = (int)sizeof(gamma_summary);
    out_host[2] = (int)sizeof(gamma_counters); out_host[3] = (int)sizeof(gamma_stage_times);
}

const char* gamma_last_error_string(void) { return g_err.c_str(); }

const char* gamma_version(void) { return "gamma_b200 0.1 sm_100a"; }

}  // extern "C"
