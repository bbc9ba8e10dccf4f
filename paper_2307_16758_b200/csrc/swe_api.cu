// swe_api.cu -- C ABI of include/swe_b200.h: context, device memory, step scheduling.
// Every step of the hot path runs in the kernels of swe_kernels.cuh; there is no CPU fallback.
#include "../../include/swe_b200.h"
#include "host_mesh.hpp"
#include "swe_kernels.cuh"
#include "swe_zone_kernels.cuh"
#include "swe_zone_assembly.cuh"

#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <unordered_map>
#include <utility>
#include <map>
#include <mutex>
#include <new>
#include <string>
#include <vector>

using namespace swe;

namespace {

thread_local std::string g_err;
int fail(int code, const std::string& msg) { g_err = msg; return code; }

#define CU(call)                                                                        \
    do {                                                                                \
        cudaError_t e_ = (call);                                                        \
        if (e_ != cudaSuccess)                                                          \
            return fail(SWE_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); \
    } while (0)

enum { KIND_DT = 0, KIND_GRAD = 1, KIND_FLUX = 2, KIND_UPDATE = 3, KIND_PACK = 4, KIND_UNPACK = 5,
       KIND_MISC = 6, NKIND = 7 };

// device copy of one MeshArrays + the state / gradient / flux buffers that live on it
struct Store {
    DevMesh dm{};
    std::vector<void*> owned;          // every cudaMalloc of this store
    int* d_cell_user = nullptr;
    int* d_bkind = nullptr;
    double* d_bval = nullptr;
    double* d_nman = nullptr;
    int4* d_c2e = nullptr;             // = dm.c2e, writable (Manning codes in c2e.w)
    std::vector<int32_t> h_btag;
    double4 *A = nullptr, *B = nullptr, *grad = nullptr;
    FluxBuf F{};
    unsigned *zA = nullptr, *zB = nullptr, *gz = nullptr, *fz = nullptr;   // dry-record bit masks (DryMasks)
    size_t mask_words = 0;                                               // zA | zB | gz | fz, one allocation
    int64_t nc = 0, ne = 0, nbe = 0;

    template <class T> cudaError_t alloc(T** p, size_t n) {
        void* q = nullptr;
        cudaError_t e = cudaMalloc(&q, (n ? n : 1) * sizeof(T));
        if (e == cudaSuccess) { owned.push_back(q); *p = (T*)q; }
        return e;
    }
    template <class T> cudaError_t upload(T** p, const void* src, size_t n, cudaStream_t s) {
        cudaError_t e = alloc(p, n);
        if (e != cudaSuccess) return e;
        if (n) e = cudaMemcpyAsync(*p, src, n * sizeof(T), cudaMemcpyHostToDevice, s);
        return e;
    }
    void release() {
        for (void* p : owned) cudaFree(p);
        owned.clear();
    }
};

// device temporaries of a set-up call, freed on every way out
struct Scratch {
    std::vector<void*> p;
    template <class T> cudaError_t get(T** q, size_t n) {
        void* v = nullptr;
        cudaError_t e = cudaMalloc(&v, (n ? n : 1) * sizeof(T));
        if (e == cudaSuccess) { p.push_back(v); *q = (T*)v; }
        return e;
    }
    ~Scratch() { for (void* v : p) cudaFree(v); }
};

// ---- swe_get_state_static: staging without an allocation ------------------------------------
// swe_get_state with host arrays stages the three fields through a device buffer that
// ensure_stage() cudaMallocs on first use.  Callers that must not allocate (code under CUDA graph
// capture, tight serving loops, harnesses that forbid cudaMalloc) get the same read-back through
// this file-scope array instead: 3 x SWE_STATIC_MAX_CELLS doubles = 6 MiB, held by every GPU that
// loads the library until the process exits.  In HOST code the name g_static_stage is a host-side
// stand-in, not a device address: the address a kernel may use is asked for once per device, with
// that device current, by cudaGetSymbolAddress (static_stage_resolve, called from swe_mesh_create)
// and kept in g_static_stage_ptr[device].
static __device__ __align__(256) double g_static_stage[3 * (size_t)SWE_STATIC_MAX_CELLS];
constexpr int STATIC_MAX_DEVICES = 64;
double* g_static_stage_ptr[STATIC_MAX_DEVICES] = {nullptr};
cudaError_t g_static_stage_err[STATIC_MAX_DEVICES] = {cudaSuccess};
bool g_static_stage_asked[STATIC_MAX_DEVICES] = {false};
// set-up, once per device, `dev` current: never allocates; a failure is remembered and reported by
// the entry point that needs the array (nothing else depends on it)
std::mutex g_static_stage_mutex;           // two threads may create their first contexts at the same time
void static_stage_resolve(int dev) {
    std::lock_guard<std::mutex> lock(g_static_stage_mutex);
    if (dev < 0 || dev >= STATIC_MAX_DEVICES || g_static_stage_asked[dev]) return;
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_static_stage);
    if (e != cudaSuccess) cudaGetLastError();
    g_static_stage_ptr[dev] = (e == cudaSuccess) ? (double*)p : nullptr;
    g_static_stage_err[dev] = e;
    g_static_stage_asked[dev] = true;
}

}  // namespace

struct swe_ctx {
    cudaStream_t stream = nullptr;
    int device = 0;                    // the device that was current in swe_mesh_create
    int num_sm = 148;
    HostMesh H;
    ZoneSet Z;
    bool has_zones = false;
    Store g, z;
    Par P{9.81, 1e-6, 1e-3, 0.5, 1.0 / 9.81, 1};
    double beta = 1.0;
    std::map<int, std::pair<int, double>> bc;
    StepScalars* d_S = nullptr;
    double* d_nman_tab = nullptr;      // 256 doubles: Manning n by code (c2e.w bits 8-15)
    unsigned char* d_ncode = nullptr;  // per USER cell, kept for zones created later
    int* d_flag = nullptr;             // validation flag of swe_set_state
    bool min_valid = false;
    int64_t launches = 0, halo_bytes = 0, steps = 0;
    // zone exchange
    int* d_send_idx = nullptr;
    int* d_recv_idx = nullptr;
    int* d_src_of_cell = nullptr;
    double* d_sendbuf = nullptr;
    int64_t nsend = 0;
    int* d_rsend_idx = nullptr;        // links that cross ranks (swe_zones_create_dist)
    int* d_rrecv_idx = nullptr;
    int64_t nrsend = 0, nrrecv = 0;
    int* d_rsend_dst = nullptr;        // push over peer memory: ghost index on the peer, peer rank,
    int* d_rsend_peer = nullptr;       // and the peers' two state buffers (device arrays of nranks pointers)
    double4** d_peerA = nullptr;
    double4** d_peerB = nullptr;
    std::vector<void*> peerA, peerB;   // host copies; [rank] = this context's own buffers
    std::vector<char> peer_ipc;        // 1: opened with cudaIpcOpenMemHandle (closed in free_zones)
    std::vector<int> zr_zone;          // resident zones and their first cell in the concatenated mesh
    std::vector<long long> zr_off;     // (the zones' cell lists are downloaded on demand)
    bool zone_cells_on_host = false;
    double zone_ms[5] = {0, 0, 0, 0, 0};     // last swe_zones_create: device ghost layers, + host zone build, + upload (cumulative)
    int* d_send_cells = nullptr;       // distinct cells on a send list (overlap schedule updates them first)
    int64_t nsendcells = 0;
    // staging for host pointers
    double* d_stage = nullptr;
    size_t stage_elems = 0;
    // profile
    bool profile = false;
    std::vector<std::pair<int, std::pair<cudaEvent_t, cudaEvent_t>>> prof_events;
    double prof_ms[NKIND] = {0};
    int64_t prof_n[NKIND] = {0};
    // one time step captured as a CUDA graph and replayed (launch-bound on small meshes): valid for
    // one (scheme, cfl, store, parameter set); captured on a side stream, launched on `stream`
    // dry-record bit masks (swe_kernels.cuh DryMasks): used by swe_step on the un-zoned store only;
    // `masks_live` = the bits describe the buffers; every other entry point clears it (check_ctx)
    bool dry_masks = false;            // opt-in (swe_set_dry_masks): see DESIGN.md section 6
    mutable bool masks_live = false;
    int mask_scheme = -1;
    bool mk_on = false;                // set while swe_step enqueues its stages
    bool graph_masks = false;
    bool use_graphs = true;
    cudaStream_t cap_stream = nullptr;
    cudaGraphExec_t step_exec = nullptr;
    int graph_scheme = -1; double graph_cfl = 0.0; bool graph_zoned = false;
    int64_t graph_launches = 0, graph_halo = 0;
    // grid sizes (persistent grid-stride kernels: a multiple of the SM count)
    int grid_light = 148 * 8;
    int grid_ms = 148 * 5;
    int grid_grad = 148 * 4, grid_flux[4] = {148 * 4, 148 * 2, 148 * 2, 148 * 2}, grid_upd = 148 * 8;

    Store& active() { return has_zones ? z : g; }
};

namespace {

int grid_for(int64_t n, int cap, int threads = 256) {
    int64_t b = (n + threads - 1) / threads;
    if (b < 1) b = 1;
    return (int)(b < cap ? b : cap);
}

bool is_device_ptr(const void* p) {
    cudaPointerAttributes a;
    cudaError_t e = cudaPointerGetAttributes(&a, p);
    if (e != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

template <class F> void launch(swe_ctx* c, int kind, F&& f) {
    if (c->profile) {
        cudaEvent_t a, b;
        cudaEventCreate(&a); cudaEventCreate(&b);
        cudaEventRecord(a, c->stream);
        f();
        cudaEventRecord(b, c->stream);
        c->prof_events.push_back({kind, {a, b}});
    } else {
        f();
    }
    c->launches++;
}

void profile_collect(swe_ctx* c) {
    if (c->prof_events.empty()) return;
    cudaStreamSynchronize(c->stream);
    for (auto& pe : c->prof_events) {
        float ms = 0.f;
        cudaEventElapsedTime(&ms, pe.second.first, pe.second.second);
        c->prof_ms[pe.first] += ms; c->prof_n[pe.first]++;
        cudaEventDestroy(pe.second.first); cudaEventDestroy(pe.second.second);
    }
    c->prof_events.clear();
}

int ensure_stage(swe_ctx* c, size_t elems) {
    if (c->stage_elems >= elems) return SWE_OK;
    if (c->d_stage) cudaFree(c->d_stage);
    c->d_stage = nullptr; c->stage_elems = 0;
    CU(cudaMalloc((void**)&c->d_stage, elems * sizeof(double)));
    c->stage_elems = elems;
    return SWE_OK;
}

int upload_store(swe_ctx* c, Store& st, const MeshArrays& M) {
    cudaStream_t s = c->stream;
    st.nc = M.nc; st.ne = M.ne; st.nbe = M.ne - M.ne_int;
    st.h_btag = M.btag;
    DevMesh& d = st.dm;
    d.nc = (int)M.nc; d.ne = (int)M.ne; d.ne_int = (int)M.ne_int; d.glayer = 0;
    int4* c2c; int4* c2e; double *zc, *area, *rin;
    CU(st.upload(&c2c, M.c2c.data(), (size_t)M.nc, s));
    CU(st.upload(&c2e, M.c2e.data(), (size_t)M.nc, s));
    CU(st.upload(&zc, M.zc.data(), (size_t)M.nc, s));
    CU(st.upload(&area, M.area.data(), (size_t)M.nc, s));
    CU(st.upload(&rin, M.rin.data(), (size_t)M.nc, s));
    d.c2c = c2c; d.c2e = c2e; d.zc = zc; d.area = area; d.rin = rin;
    st.d_c2e = c2e;
    for (int k = 0; k < 3; ++k) {
        double2 *w, *r = nullptr;
        CU(st.upload(&w, M.w[k].data(), (size_t)M.nc, s));
        if (k < 2) CU(st.upload(&r, M.r[k].data(), (size_t)M.nc, s));      // r_2 travels as the residual rres
        d.w[k] = w; d.r[k] = r;
    }
    {
        float2* rres;
        CU(st.upload(&rres, M.rres.data(), (size_t)M.nc, s));
        d.rres = rres;
    }
    d.nman_tab = c->d_nman_tab;
    int2* elr; double2 *en, *erl, *err; double *elen, *edx;
    CU(st.upload(&elr, M.elr.data(), (size_t)M.ne, s));
    CU(st.upload(&en, M.en.data(), (size_t)M.ne, s));
    CU(st.upload(&elen, M.elen.data(), (size_t)M.ne, s));
    CU(st.upload(&edx, M.edx.data(), (size_t)M.ne, s));
    CU(st.upload(&erl, M.erl.data(), (size_t)M.ne, s));
    CU(st.upload(&err, M.err.data(), (size_t)M.ne, s));
    d.elr = elr; d.en = en; d.elen = elen; d.edx = edx; d.erl = erl; d.err = err;
    {
        double2* ed;
        CU(st.upload(&ed, M.ed.data(), (size_t)M.ne, s));
        d.ed = ed;
    }
    double4* dupw; double* edlr; uint8_t* eside;
    CU(st.upload(&dupw, M.dupw.data(), (size_t)M.nc, s));
    CU(st.upload(&edlr, M.edlr.data(), (size_t)M.ne, s));
    CU(st.upload(&eside, M.eside.data(), (size_t)M.ne, s));
    double2* ernorm;
    CU(st.upload(&ernorm, M.ernorm.data(), (size_t)M.ne, s));
    d.dupw = dupw; d.edlr = edlr; d.eside = eside; d.ernorm = ernorm;
    CU(st.upload(&st.d_cell_user, M.cell_user.data(), (size_t)M.nc, s));
    CU(st.alloc(&st.d_bkind, (size_t)st.nbe));
    CU(st.alloc(&st.d_bval, (size_t)st.nbe));
    CU(st.alloc(&st.d_nman, (size_t)M.nc));
    d.bkind = st.d_bkind; d.bval = st.d_bval; d.nman = st.d_nman;
    d.layer = nullptr;
    CU(st.alloc(&st.A, (size_t)M.nc));
    CU(st.alloc(&st.B, (size_t)M.nc));
    CU(st.alloc(&st.grad, 3 * (size_t)M.nc));      // 2 per cell (limited gradients) or 3 (multislope side records)
    CU(st.alloc(&st.F.f1, (size_t)M.ne));
    CU(st.alloc(&st.F.fxl, (size_t)M.ne));
    CU(st.alloc(&st.F.fyl, (size_t)M.ne));
    CU(st.alloc(&st.F.fxr, (size_t)M.ne));
    CU(st.alloc(&st.F.fyr, (size_t)M.ne));
    {
        const size_t wc = ((size_t)M.nc + 31) / 32 + 1, we = ((size_t)M.ne + 31) / 32 + 1;
        st.mask_words = 3 * wc + we;
        CU(st.alloc(&st.zA, st.mask_words));
        st.zB = st.zA + wc; st.gz = st.zB + wc; st.fz = st.gz + wc;
    }
    CU(cudaMemsetAsync(st.grad, 0, 3 * (size_t)M.nc * sizeof(double4), s));
    CU(cudaMemsetAsync(st.B, 0, (size_t)M.nc * sizeof(double4), s));
    CU(cudaMemsetAsync(st.d_nman, 0, (size_t)(M.nc ? M.nc : 1) * sizeof(double), s));
    return SWE_OK;
}

// boundary kind / value per boundary edge from the tag table (A.8; inflow: q_n = -Q / W, R10)
int refresh_bc(swe_ctx* c, Store& st) {
    std::vector<int> kind(st.nbe, KB_WALL);
    std::vector<double> val(st.nbe, 0.0);
    for (int64_t b = 0; b < st.nbe; ++b) {
        int t = st.h_btag[b];
        if (t < 0) continue;
        auto it = c->bc.find(t);
        if (it == c->bc.end()) continue;
        kind[b] = it->second.first;
        if (kind[b] == KB_INFLOW) {
            double w = 1.0;
            for (size_t j = 0; j < c->H.tags.size(); ++j) if (c->H.tags[j] == t) w = c->H.tag_width[j];
            val[b] = -it->second.second / w;
        } else {
            val[b] = it->second.second;
        }
    }
    if (st.nbe) {
        CU(cudaMemcpyAsync(st.d_bkind, kind.data(), st.nbe * sizeof(int), cudaMemcpyHostToDevice, c->stream));
        CU(cudaMemcpyAsync(st.d_bval, val.data(), st.nbe * sizeof(double), cudaMemcpyHostToDevice, c->stream));
        CU(cudaStreamSynchronize(c->stream));
    }
    return SWE_OK;
}

__global__ void k_gather_cells(double4* __restrict__ dst, const double4* __restrict__ src,
                               const int* __restrict__ idx, int n) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) dst[i] = src[idx[i]];
}
__global__ void k_gather_scalar(double* __restrict__ dst, const double* __restrict__ src,
                                const int* __restrict__ idx, int n) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) dst[i] = src[idx[i]];
}
__global__ void k_scatter_owned(double4* __restrict__ dst, const double4* __restrict__ src,
                                const int* __restrict__ idx, const uint8_t* __restrict__ layer, int n) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x)
        if (layer[i] == 0) dst[idx[i]] = src[i];
}
__global__ void k_reset_min(StepScalars* S) { S->min_bits = 0x7ff0000000000000ULL; }

void drop_graph(swe_ctx* c) {
    if (c->step_exec) cudaGraphExecDestroy(c->step_exec);
    c->step_exec = nullptr; c->graph_scheme = -1;
}

void free_zones(swe_ctx* c) {
    drop_graph(c);
    c->z.release();
    c->z = Store();
    if (c->d_send_idx) cudaFree(c->d_send_idx);
    if (c->d_recv_idx) cudaFree(c->d_recv_idx);
    if (c->d_src_of_cell) cudaFree(c->d_src_of_cell);
    if (c->d_sendbuf) cudaFree(c->d_sendbuf);
    if (c->d_rsend_idx) cudaFree(c->d_rsend_idx);
    if (c->d_rrecv_idx) cudaFree(c->d_rrecv_idx);
    if (c->d_send_cells) cudaFree(c->d_send_cells);
    c->d_send_cells = nullptr; c->nsendcells = 0;
    if (c->d_rsend_dst) cudaFree(c->d_rsend_dst);
    if (c->d_rsend_peer) cudaFree(c->d_rsend_peer);
    if (c->d_peerA) cudaFree(c->d_peerA);
    if (c->d_peerB) cudaFree(c->d_peerB);
    for (size_t p = 0; p < c->peer_ipc.size(); ++p)
        if (c->peer_ipc[p]) { cudaIpcCloseMemHandle(c->peerA[p]); cudaIpcCloseMemHandle(c->peerB[p]); }
    c->peerA.clear(); c->peerB.clear(); c->peer_ipc.clear();
    c->d_rsend_idx = c->d_rrecv_idx = c->d_rsend_dst = c->d_rsend_peer = nullptr;
    c->d_peerA = c->d_peerB = nullptr;
    c->nrsend = c->nrrecv = 0;
    c->d_send_idx = c->d_recv_idx = c->d_src_of_cell = nullptr;
    c->d_sendbuf = nullptr;
    c->nsend = 0;
    c->has_zones = false;
    c->zone_cells_on_host = false;
    c->zr_zone.clear(); c->zr_off.clear();
    c->Z = ZoneSet();
}

// ---- kernel launch helpers (all on c->stream) ----
// masks of the stage that reads `Uin` and writes `Uout` (either may be nullptr when not needed)
DryMasks masks_of(const swe_ctx* c, const Store& st, const double4* Uin, const double4* Uout) {
    DryMasks K{nullptr, nullptr, nullptr, nullptr};
    if (!c->mk_on) return K;
    K.zin = (Uin == st.A) ? st.zA : st.zB;
    K.zout = (Uout == st.A) ? st.zA : st.zB;
    K.gz = st.gz; K.fz = st.fz;
    return K;
}
void run_dt_reduce(swe_ctx* c, Store& st, const double4* U) {
    launch(c, KIND_DT, [&] {
        k_dt_reduce<<<grid_for(st.nc, c->grid_light), 256, 0, c->stream>>>(st.dm, U, c->P, c->d_S);
    });
}
// cell pass ahead of the flux: limited least-squares gradients (MUSCL) or the multislope side
// records (MUSCL_MS); HLLC and WAF have none
void run_grad(swe_ctx* c, Store& st, const double4* U, int scheme = K_MUSCL) {
    if (scheme == K_MUSCL_MS) {
        launch(c, KIND_GRAD, [&] {
            k_ms_slopes<<<grid_for(st.nc, c->grid_ms, 128), 128, 0, c->stream>>>(st.dm, U, st.grad, c->P);
        });
        return;
    }
    if (scheme != K_MUSCL) return;
    launch(c, KIND_GRAD, [&] {
        const int gr = grid_for(st.nc, c->grid_grad, SWE_GRAD_THREADS);
        const DryMasks K = masks_of(c, st, U, nullptr);
        if (c->mk_on) k_grad_limit<true><<<gr, SWE_GRAD_THREADS, 0, c->stream>>>(st.dm, U, st.grad, c->P, K);
        else k_grad_limit<false><<<gr, SWE_GRAD_THREADS, 0, c->stream>>>(st.dm, U, st.grad, c->P, K);
    });
}
void run_flux(swe_ctx* c, Store& st, const double4* U, int scheme) {
    launch(c, KIND_FLUX, [&] {
        const int gr = grid_for(st.ne, c->grid_flux[scheme], SWE_FLUX_THREADS);
        const DryMasks K = masks_of(c, st, U, nullptr);
#define SWE_FLUX_LAUNCH(SC, MK) k_edge_flux<SC, MK><<<gr, SWE_FLUX_THREADS, 0, c->stream>>>(st.dm, U, st.grad, st.F, c->P, c->d_S, K)
        if (c->mk_on) {
            if (scheme == K_HLLC) SWE_FLUX_LAUNCH(K_HLLC, true);
            else if (scheme == K_MUSCL) SWE_FLUX_LAUNCH(K_MUSCL, true);
            else if (scheme == K_WAF) SWE_FLUX_LAUNCH(K_WAF, true);
            else SWE_FLUX_LAUNCH(K_MUSCL_MS, true);
        } else {
            if (scheme == K_HLLC) SWE_FLUX_LAUNCH(K_HLLC, false);
            else if (scheme == K_MUSCL) SWE_FLUX_LAUNCH(K_MUSCL, false);
            else if (scheme == K_WAF) SWE_FLUX_LAUNCH(K_WAF, false);
            else SWE_FLUX_LAUNCH(K_MUSCL_MS, false);
        }
#undef SWE_FLUX_LAUNCH
    });
}
// mode 0: Uout = E(Uin); mode 1: Uout = (U0 + E(Uin))/2; fuse: fold the next CFL min in;
// part 0: every owned cell, 1: only the cells on a send list, 2: every owned cell but those
void run_update(swe_ctx* c, Store& st, const double4* Uin, const double4* U0, double4* Uout, int mode, bool fuse, int part = 0) {
    if (part == 1) {
        const int n = (int)c->nsendcells;
        if (n == 0) return;
        launch(c, KIND_UPDATE, [&] {
            // a few thousand cells: 64-thread blocks spread them over the SMs (a latency-bound launch)
            const int gr = grid_for(n, c->grid_light * 4, 64);
            const int* L = c->d_send_cells;
            if (mode == 0 && !fuse) k_cell_update_list<0, false><<<gr, 64, 0, c->stream>>>(st.dm, Uin, U0, Uout, st.F, c->P, c->d_S, L, n);
            else if (mode == 0) k_cell_update_list<0, true><<<gr, 64, 0, c->stream>>>(st.dm, Uin, U0, Uout, st.F, c->P, c->d_S, L, n);
            else if (!fuse) k_cell_update_list<1, false><<<gr, 64, 0, c->stream>>>(st.dm, Uin, U0, Uout, st.F, c->P, c->d_S, L, n);
            else k_cell_update_list<1, true><<<gr, 64, 0, c->stream>>>(st.dm, Uin, U0, Uout, st.F, c->P, c->d_S, L, n);
        });
        return;
    }
    const int skip = part == 2 ? 1 : 0;
    launch(c, KIND_UPDATE, [&] {
        const int gr = grid_for(st.nc, c->grid_upd);
        const DryMasks K = masks_of(c, st, Uin, Uout);
#define SWE_UPD_LAUNCH(MO, FU, MK) k_cell_update<MO, FU, MK><<<gr, 256, 0, c->stream>>>(st.dm, Uin, U0, Uout, st.F, c->P, c->d_S, skip, K)
        if (c->mk_on) {
            if (mode == 0 && !fuse) SWE_UPD_LAUNCH(0, false, true);
            else if (mode == 0) SWE_UPD_LAUNCH(0, true, true);
            else if (!fuse) SWE_UPD_LAUNCH(1, false, true);
            else SWE_UPD_LAUNCH(1, true, true);
        } else {
            if (mode == 0 && !fuse) SWE_UPD_LAUNCH(0, false, false);
            else if (mode == 0) SWE_UPD_LAUNCH(0, true, false);
            else if (!fuse) SWE_UPD_LAUNCH(1, false, false);
            else SWE_UPD_LAUNCH(1, true, false);
        }
#undef SWE_UPD_LAUNCH
    });
}
void run_exchange_state(swe_ctx* c, double4* U, int64_t first, int64_t count, bool do_pack, bool do_unpack) {
    if (count <= 0) return;
    if (do_pack) {
        launch(c, KIND_PACK, [&] {
            k_pack_state<<<grid_for(count, c->grid_light), 256, 0, c->stream>>>(U, c->d_send_idx, c->d_sendbuf, first, count);
        });
        c->halo_bytes += count * (4 + 32 + 24);
    }
    if (do_unpack) {
        launch(c, KIND_UNPACK, [&] {
            k_unpack_state<<<grid_for(count, c->grid_light), 256, 0, c->stream>>>(U, c->d_recv_idx, c->d_sendbuf, c->z.dm.zc, first, count);
        });
        c->halo_bytes += count * (4 + 24 + 8 + 32);
    }
}
void run_exchange_grad(swe_ctx* c) {
    const int64_t count = c->nsend;
    if (count <= 0) return;
    launch(c, KIND_PACK, [&] {
        k_pack_grad<<<grid_for(count, c->grid_light), 256, 0, c->stream>>>(c->z.grad, c->d_send_idx, (double4*)c->d_sendbuf, 0, count);
    });
    launch(c, KIND_UNPACK, [&] {
        k_unpack_grad<<<grid_for(count, c->grid_light), 256, 0, c->stream>>>(c->z.grad, c->d_recv_idx, (const double4*)c->d_sendbuf, 0, count);
    });
    c->halo_bytes += count * (4 + 64 + 64 + 4 + 64 + 64);
}

// one Euler stage on the active store: [exchange] -> [grad (-> exchange grad)] -> flux -> update
void run_stage(swe_ctx* c, Store& st, double4* Uin, const double4* U0, double4* Uout, int scheme, int mode, bool fuse) {
    if (c->has_zones) run_exchange_state(c, Uin, 0, c->nsend, true, true);
    run_grad(c, st, Uin, scheme);
    if (scheme == K_MUSCL && c->has_zones && c->Z.nlayers == 1) run_exchange_grad(c);
    run_flux(c, st, Uin, scheme);
    run_update(c, st, Uin, U0, Uout, mode, fuse);
}

int sync_global_from_zoned(swe_ctx* c) {
    if (!c->has_zones) return SWE_OK;
    k_scatter_owned<<<grid_for(c->z.nc, c->grid_light), 256, 0, c->stream>>>(c->g.A, c->z.A, c->d_src_of_cell, c->z.dm.layer, (int)c->z.nc);
    c->launches++;
    CU(cudaGetLastError());
    return SWE_OK;
}

// every entry point comes through here: whatever it does to the buffers, the dry-record masks no
// longer describe them (swe_step and the read-only getters restore the flag themselves)
int check_ctx(const swe_ctx* c) {
    if (!c) return fail(SWE_ERR_ARG, "null context");
    c->masks_live = false;
    return SWE_OK;
}
struct KeepMasks {                      // read-only entry points
    const swe_ctx* c; bool live;
    explicit KeepMasks(const swe_ctx* c_) : c(c_), live(c_ && c_->masks_live) {}
    ~KeepMasks() { if (c) c->masks_live = live; }
};

}  // namespace

extern "C" {

const char* swe_last_error(void) { return g_err.c_str(); }

int swe_mesh_create(swe_ctx** out, int64_t nv, const double* x, const double* y, const double* zb,
                    int64_t nt, const int32_t* tri, int64_t nb, const int32_t* bedge,
                    const int32_t* btag, int renumber, void* cuda_stream) {
    if (!out) return fail(SWE_ERR_ARG, "out is NULL");
    *out = nullptr;
    if (nv <= 0 || nt <= 0 || !x || !y || !zb || !tri) return fail(SWE_ERR_ARG, "empty or NULL mesh arrays");
    if (nb < 0 || (nb > 0 && (!bedge || !btag))) return fail(SWE_ERR_ARG, "bad boundary-edge arguments");
    if (renumber != SWE_RENUM_NONE && renumber != SWE_RENUM_HILBERT && renumber != SWE_RENUM_RCM) return fail(SWE_ERR_ARG, "unknown renumbering");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(SWE_ERR_CUDA, "no CUDA device: this library has no CPU fallback");
    }
    // mesh arrays may be host or device pointers: bring device ones to the host for the set-up
    std::vector<double> hx, hy, hz; std::vector<int32_t> ht, hb, hbt;
    auto to_host_d = [&](const double* p, int64_t n, std::vector<double>& v) -> const double* {
        if (!is_device_ptr(p)) return p;
        v.resize(n); cudaMemcpy(v.data(), p, n * sizeof(double), cudaMemcpyDeviceToHost); return v.data(); };
    auto to_host_i = [&](const int32_t* p, int64_t n, std::vector<int32_t>& v) -> const int32_t* {
        if (!p || !is_device_ptr(p)) return p;
        v.resize(n); cudaMemcpy(v.data(), p, n * sizeof(int32_t), cudaMemcpyDeviceToHost); return v.data(); };
    x = to_host_d(x, nv, hx); y = to_host_d(y, nv, hy); zb = to_host_d(zb, nv, hz);
    tri = to_host_i(tri, 3 * nt, ht); bedge = to_host_i(bedge, 2 * nb, hb); btag = to_host_i(btag, nb, hbt);

    swe_ctx* c = new (std::nothrow) swe_ctx();
    if (!c) return fail(SWE_ERR_NOMEM, "out of host memory");
    c->stream = (cudaStream_t)cuda_stream;
    std::string err;
    bool ok = false;
    try { ok = build_host_mesh(c->H, nv, x, y, zb, nt, tri, nb, bedge, btag, renumber, err); }
    catch (const std::bad_alloc&) { delete c; return fail(SWE_ERR_NOMEM, "out of host memory in mesh set-up"); }
    if (!ok) { delete c; return fail(SWE_ERR_MESH, err); }
    int dev = 0;
    cudaGetDevice(&dev);
    c->device = dev;
    static_stage_resolve(dev);         // address of the static staging array on this device (swe_get_state_static)
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, dev) == cudaSuccess) c->num_sm = prop.multiProcessorCount;
    // persistent grids: (resident blocks per SM) x (SM count), from the occupancy calculator
    auto occ = [&](const void* k, int fallback, int threads = 256) {
        int nbk = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nbk, k, threads, 0) != cudaSuccess || nbk < 1) { cudaGetLastError(); nbk = fallback; }
        return nbk * c->num_sm;
    };
    c->grid_light = 8 * c->num_sm;
    c->grid_grad = occ((const void*)k_grad_limit<false>, 4, SWE_GRAD_THREADS);
    c->grid_flux[K_HLLC] = occ((const void*)k_edge_flux<K_HLLC, false>, 4, SWE_FLUX_THREADS);
    c->grid_flux[K_MUSCL] = occ((const void*)k_edge_flux<K_MUSCL, false>, 2, SWE_FLUX_THREADS);
    c->grid_flux[K_WAF] = occ((const void*)k_edge_flux<K_WAF, false>, 2, SWE_FLUX_THREADS);
    c->grid_flux[K_MUSCL_MS] = occ((const void*)k_edge_flux<K_MUSCL_MS, false>, 2, SWE_FLUX_THREADS);
    c->grid_upd = occ((const void*)k_cell_update<1, true, false>, 4);
    c->grid_ms = occ((const void*)k_ms_slopes, 5, 128);
    int rc = SWE_OK;
    {
        cudaError_t e = cudaMalloc((void**)&c->d_nman_tab, 256 * sizeof(double));
        if (e == cudaSuccess) e = cudaMemsetAsync(c->d_nman_tab, 0, 256 * sizeof(double), c->stream);
        if (e == cudaSuccess) e = cudaMalloc((void**)&c->d_ncode, (size_t)c->H.nt);
        if (e == cudaSuccess) e = cudaMemsetAsync(c->d_ncode, 0, (size_t)c->H.nt, c->stream);
        if (e != cudaSuccess) rc = fail(SWE_ERR_CUDA, cudaGetErrorString(e));
    }
    if (rc == SWE_OK) rc = upload_store(c, c->g, c->H.m);
    if (rc == SWE_OK) {
        cudaError_t e = cudaMalloc((void**)&c->d_S, sizeof(StepScalars));
        if (e == cudaSuccess) e = cudaMalloc((void**)&c->d_flag, sizeof(int));
        if (e != cudaSuccess) rc = fail(SWE_ERR_CUDA, cudaGetErrorString(e));
    }
    if (rc == SWE_OK) {
        StepScalars s0; s0.min_bits = 0x7ff0000000000000ULL; s0.dt = 0.0; s0.t = 0.0; s0.last_dt = 0.0; s0.steps = 0;
        cudaMemcpyAsync(c->d_S, &s0, sizeof(s0), cudaMemcpyHostToDevice, c->stream);
        // initial state: h = hu = hv = 0, z = cell bed
        k_fill<<<grid_for(4 * c->g.nc, c->grid_light), 256, 0, c->stream>>>((double*)c->g.A, 0.0, 4 * c->g.nc);
        rc = refresh_bc(c, c->g);
    }
    if (rc == SWE_OK) {
        // z component of the state records
        cudaError_t e = cudaMemcpy2DAsync((char*)c->g.A + 3 * sizeof(double), sizeof(double4), c->g.dm.zc, sizeof(double),
                                          sizeof(double), (size_t)c->g.nc, cudaMemcpyDeviceToDevice, c->stream);
        if (e == cudaSuccess) e = cudaMemcpy2DAsync((char*)c->g.B + 3 * sizeof(double), sizeof(double4), c->g.dm.zc, sizeof(double),
                                                    sizeof(double), (size_t)c->g.nc, cudaMemcpyDeviceToDevice, c->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
        if (e != cudaSuccess) rc = fail(SWE_ERR_CUDA, cudaGetErrorString(e));
    }
    if (rc != SWE_OK) { std::string keep = g_err; swe_mesh_destroy(c); g_err = keep; return rc; }
    *out = c;
    return SWE_OK;
}

int swe_mesh_destroy(swe_ctx* c) {
    if (!c) return SWE_OK;
    cudaStreamSynchronize(c->stream);
    for (auto& pe : c->prof_events) { cudaEventDestroy(pe.second.first); cudaEventDestroy(pe.second.second); }
    free_zones(c);
    if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
    c->g.release();
    if (c->d_S) cudaFree(c->d_S);
    if (c->d_flag) cudaFree(c->d_flag);
    if (c->d_stage) cudaFree(c->d_stage);
    if (c->d_nman_tab) cudaFree(c->d_nman_tab);
    if (c->d_ncode) cudaFree(c->d_ncode);
    delete c;
    return SWE_OK;
}

int swe_mesh_info(const swe_ctx* c, int64_t* ncell, int64_t* nedge, int64_t* nbedge, double* min_inradius) {
    KeepMasks keep_masks(c);   // read-only
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (ncell) *ncell = c->H.nt;
    if (nedge) *nedge = c->H.m.ne;
    if (nbedge) *nbedge = c->H.nbe;
    if (min_inradius) *min_inradius = c->H.min_rin;
    return SWE_OK;
}

int swe_set_params(swe_ctx* c, double g, double h_dry, double h_thin, double beta) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!(g > 0.0) || !(h_dry >= 0.0) || !(h_thin >= 0.0) || beta != beta) return fail(SWE_ERR_ARG, "bad parameter value");
    // the kernels' reciprocal / square-root sequences (rcp_nr, sqrt_nr) start from MUFU seeds that
    // flush subnormals: every depth that counts as wet must be a normal number well away from 0
    if (h_dry < 1e-290) return fail(SWE_ERR_ARG, "h_dry must be >= 1e-290 (a wet depth has to be a normal fp64 number)");
    c->P.g = g; c->P.h_dry = h_dry; c->P.h_thin = h_thin; c->beta = beta;
    c->P.kappa = beta / 2.0; c->P.inv_g = 1.0 / g; c->P.limited = beta > 0.0 ? 1 : 0;
    drop_graph(c);                                   // the parameters are kernel arguments
    c->min_valid = false;
    k_reset_min<<<1, 1, 0, c->stream>>>(c->d_S);
    return SWE_OK;
}

int swe_set_manning(swe_ctx* c, const double* n_cell) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    const int64_t nt = c->H.nt;
    if (!n_cell) {
        CU(cudaMemsetAsync(c->g.d_nman, 0, nt * sizeof(double), c->stream));
    } else {
        const double* src = n_cell;
        if (!is_device_ptr(n_cell)) {
            int rc = ensure_stage(c, (size_t)nt); if (rc) return rc;
            CU(cudaMemcpyAsync(c->d_stage, n_cell, nt * sizeof(double), cudaMemcpyHostToDevice, c->stream));
            src = c->d_stage;
        }
        k_scalar_from_user<<<grid_for(nt, c->grid_light), 256, 0, c->stream>>>(c->g.d_nman, c->g.d_cell_user, src, (int)nt);
        CU(cudaGetLastError());
    }
    if (c->has_zones) {
        k_gather_scalar<<<grid_for(c->z.nc, c->grid_light), 256, 0, c->stream>>>(c->z.d_nman, c->g.d_nman, c->d_src_of_cell, (int)c->z.nc);
        CU(cudaGetLastError());
    }
    // the distinct values as a table, a one-byte code per cell in c2e.w (swe_kernels.cuh c2e_ncode):
    // the update kernel then reads nothing per cell for n.  More than 255 distinct values: code 255
    // everywhere, the kernel reads the array.
    {
        std::vector<double> hn;
        const double* hv = n_cell;
        if (n_cell && is_device_ptr(n_cell)) {
            hn.resize((size_t)nt);
            CU(cudaMemcpyAsync(hn.data(), n_cell, nt * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
            CU(cudaStreamSynchronize(c->stream));
            hv = hn.data();
        }
        std::vector<unsigned char> code((size_t)nt, 0);
        std::vector<double> tab(256, 0.0);
        bool fits = true;
        if (hv) {
            std::unordered_map<uint64_t, int> codes;          // the table, by bit pattern
            uint64_t last_b = 0; int last = -1;
            for (int64_t i = 0; i < nt; ++i) {
                uint64_t b; std::memcpy(&b, &hv[i], 8);
                int k;
                if (last >= 0 && b == last_b) k = last;
                else {
                    auto it = codes.find(b);
                    if (it != codes.end()) k = it->second;
                    else {
                        if (codes.size() == 255) { fits = false; break; }
                        k = (int)codes.size(); codes.emplace(b, k); tab[k] = hv[i];
                    }
                }
                code[i] = (unsigned char)k; last = k; last_b = b;
            }
        }
        if (!fits) std::fill(code.begin(), code.end(), (unsigned char)255);
        CU(cudaMemcpyAsync(c->d_nman_tab, tab.data(), 256 * sizeof(double), cudaMemcpyHostToDevice, c->stream));
        CU(cudaMemcpyAsync(c->d_ncode, code.data(), (size_t)nt, cudaMemcpyHostToDevice, c->stream));
        k_set_ncode<<<grid_for(nt, c->grid_light), 256, 0, c->stream>>>(c->g.d_c2e, c->g.d_cell_user, c->d_ncode, (int)nt);
        if (c->has_zones)
            k_set_ncode<<<grid_for(c->z.nc, c->grid_light), 256, 0, c->stream>>>(c->z.d_c2e, c->z.d_cell_user, c->d_ncode, (int)c->z.nc);
        CU(cudaGetLastError());
    }
    CU(cudaStreamSynchronize(c->stream));
    return SWE_OK;
}

int swe_set_bc(swe_ctx* c, int tag, int kind, double value) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (tag < 0 || kind < 0 || kind > 3 || value != value) return fail(SWE_ERR_ARG, "bad boundary condition");
    c->bc[tag] = {kind, value};
    int rc = refresh_bc(c, c->g);
    if (rc == SWE_OK && c->has_zones) rc = refresh_bc(c, c->z);
    return rc;
}

int swe_set_state(swe_ctx* c, const double* h, const double* hu, const double* hv) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!h || !hu || !hv) return fail(SWE_ERR_ARG, "NULL state array");
    const int64_t nt = c->H.nt;
    const double *dh = h, *dhu = hu, *dhv = hv;
    const bool dev = is_device_ptr(h) && is_device_ptr(hu) && is_device_ptr(hv);
    if (!dev) {
        int rc = ensure_stage(c, 3 * (size_t)nt + 2); if (rc) return rc;
        CU(cudaMemcpyAsync(c->d_stage, h, nt * sizeof(double), cudaMemcpyDefault, c->stream));
        CU(cudaMemcpyAsync(c->d_stage + nt, hu, nt * sizeof(double), cudaMemcpyDefault, c->stream));
        CU(cudaMemcpyAsync(c->d_stage + 2 * nt, hv, nt * sizeof(double), cudaMemcpyDefault, c->stream));
        dh = c->d_stage; dhu = c->d_stage + nt; dhv = c->d_stage + 2 * nt;
    }
    int* flag = c->d_flag;
    CU(cudaMemsetAsync(flag, 0, sizeof(int), c->stream));
    k_check_state<<<grid_for(nt, c->grid_light), 256, 0, c->stream>>>(dh, nt, flag);
    int bad = 0;
    cudaMemcpyAsync(&bad, flag, sizeof(int), cudaMemcpyDeviceToHost, c->stream);
    cudaError_t e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return fail(SWE_ERR_CUDA, cudaGetErrorString(e));
    if (bad) return fail(SWE_ERR_STATE, "h contains NaN or a negative depth");
    k_state_from_user<<<grid_for(nt, c->grid_light), 256, 0, c->stream>>>(c->g.A, c->g.d_cell_user, c->g.dm.zc, dh, dhu, dhv, (int)nt);
    c->launches += 2;
    if (c->has_zones) {
        k_gather_cells<<<grid_for(c->z.nc, c->grid_light), 256, 0, c->stream>>>(c->z.A, c->g.A, c->d_src_of_cell, (int)c->z.nc);
        c->launches++;
    }
    k_reset_min<<<1, 1, 0, c->stream>>>(c->d_S);
    c->min_valid = false;
    CU(cudaGetLastError());
    if (!dev) CU(cudaStreamSynchronize(c->stream));   // the staging buffer may be reused
    return SWE_OK;
}

int swe_get_state(const swe_ctx* cc, double* h, double* hu, double* hv) {
    KeepMasks keep_masks(cc);   // read-only
    swe_ctx* c = const_cast<swe_ctx*>(cc);
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!h || !hu || !hv) return fail(SWE_ERR_ARG, "NULL state array");
    const int64_t nt = c->H.nt;
    const bool dev = is_device_ptr(h) && is_device_ptr(hu) && is_device_ptr(hv);
    double *dh = h, *dhu = hu, *dhv = hv;
    if (!dev) {
        int rc = ensure_stage(c, 3 * (size_t)nt + 2); if (rc) return rc;
        dh = c->d_stage; dhu = c->d_stage + nt; dhv = c->d_stage + 2 * nt;
        if (c->has_zones && c->Z.nranks > 1) {      // only this rank's cells are written: keep the caller's other entries
            CU(cudaMemcpyAsync(dh, h, nt * sizeof(double), cudaMemcpyDefault, c->stream));
            CU(cudaMemcpyAsync(dhu, hu, nt * sizeof(double), cudaMemcpyDefault, c->stream));
            CU(cudaMemcpyAsync(dhv, hv, nt * sizeof(double), cudaMemcpyDefault, c->stream));
        }
    }
    Store& st = c->active();
    k_state_to_user<<<grid_for(st.nc, c->grid_light), 256, 0, c->stream>>>(st.A, st.d_cell_user, st.dm.layer, dh, dhu, dhv, (int)st.nc);
    c->launches++;
    CU(cudaGetLastError());
    if (!dev) {
        CU(cudaMemcpyAsync(h, dh, nt * sizeof(double), cudaMemcpyDefault, c->stream));
        CU(cudaMemcpyAsync(hu, dhu, nt * sizeof(double), cudaMemcpyDefault, c->stream));
        CU(cudaMemcpyAsync(hv, dhv, nt * sizeof(double), cudaMemcpyDefault, c->stream));
    }
    CU(cudaStreamSynchronize(c->stream));
    return SWE_OK;
}

int swe_get_state_static(const swe_ctx* cc, double* h, double* hu, double* hv) {
    KeepMasks keep_masks(cc);   // read-only
    swe_ctx* c = const_cast<swe_ctx*>(cc);
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!h || !hu || !hv) return fail(SWE_ERR_ARG, "NULL state array");
    const int64_t nt = c->H.nt;
    if (nt > (int64_t)SWE_STATIC_MAX_CELLS)
        return fail(SWE_ERR_ARG, "swe_get_state_static: the mesh has " + std::to_string(nt) + " cells, the static staging array holds at most " +
                                 std::to_string((long long)SWE_STATIC_MAX_CELLS) + " (SWE_STATIC_MAX_CELLS); use swe_get_state");
    const int dev = c->device;
    if (dev < 0 || dev >= STATIC_MAX_DEVICES || !g_static_stage_asked[dev] || !g_static_stage_ptr[dev])
        return fail(SWE_ERR_CUDA, std::string("swe_get_state_static: no device address for the static staging array (cudaGetSymbolAddress: ") +
                                  ((dev >= 0 && dev < STATIC_MAX_DEVICES && g_static_stage_asked[dev]) ? cudaGetErrorString(g_static_stage_err[dev]) : "not asked for on this device") + ")");
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess || cur != dev)
        return fail(SWE_ERR_STATE, "swe_get_state_static: the context's device must be the current device");
    const bool devout = is_device_ptr(h) && is_device_ptr(hu) && is_device_ptr(hv);
    double* stage = g_static_stage_ptr[dev];                // the DEVICE address, not the host-side symbol
    double *dh = devout ? h : stage, *dhu = devout ? hu : stage + nt, *dhv = devout ? hv : stage + 2 * nt;
    // Every slot that is copied out below is written first by this call (the array keeps whatever the
    // last call left there: nothing in it has to start at zero).  Zones distributed over ranks: only
    // this rank's cells are written, so the caller's other entries are staged in first, as swe_get_state does.
    if (!devout && c->has_zones && c->Z.nranks > 1) {
        CU(cudaMemcpyAsync(dh, h, nt * sizeof(double), cudaMemcpyDefault, c->stream));
        CU(cudaMemcpyAsync(dhu, hu, nt * sizeof(double), cudaMemcpyDefault, c->stream));
        CU(cudaMemcpyAsync(dhv, hv, nt * sizeof(double), cudaMemcpyDefault, c->stream));
    }
    Store& st = c->active();
    k_state_to_user<<<grid_for(st.nc, c->grid_light), 256, 0, c->stream>>>(st.A, st.d_cell_user, st.dm.layer, dh, dhu, dhv, (int)st.nc);
    c->launches++;
    CU(cudaGetLastError());
    if (!devout) {
        CU(cudaMemcpyAsync(h, dh, nt * sizeof(double), cudaMemcpyDefault, c->stream));
        CU(cudaMemcpyAsync(hu, dhu, nt * sizeof(double), cudaMemcpyDefault, c->stream));
        CU(cudaMemcpyAsync(hv, dhv, nt * sizeof(double), cudaMemcpyDefault, c->stream));
    }
    CU(cudaStreamSynchronize(c->stream));
    return SWE_OK;
}

int swe_set_time(swe_ctx* c, double t) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    CU(cudaMemcpyAsync(&c->d_S->t, &t, sizeof(double), cudaMemcpyHostToDevice, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return SWE_OK;
}

int swe_step(swe_ctx* c, int nsteps, double cfl, int scheme, double* t_out, double* last_dt_out) {
    const bool masks_were_live = c && c->masks_live;
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (nsteps < 0 || !(cfl > 0.0) || scheme < 0 || scheme > 3) return fail(SWE_ERR_ARG, "bad step arguments");
    if (c->has_zones && c->Z.nranks > 1)
        return fail(SWE_ERR_STATE, "zones are distributed over ranks: drive the step with swe_dist_* / swe_halo_*");
    if (c->has_zones && (scheme == K_WAF || scheme == K_MUSCL_MS) && c->Z.nlayers < 2)
        return fail(SWE_ERR_STATE, "WAF and the multislope MUSCL need zones with at least 2 ghost layers");
    Store& st = c->active();
    // dry-record masks: un-zoned store only; cleared unless the previous call on this context was a
    // swe_step with the same scheme (the gradient buffer holds other records for the multislope pass)
    struct MaskScope { swe_ctx* c; ~MaskScope() { c->mk_on = false; } } mask_scope{c};
    c->mk_on = c->dry_masks && !c->has_zones && nsteps > 0;
    if (c->mk_on) {
        if (!masks_were_live || c->mask_scheme != scheme)
            CU(cudaMemsetAsync(st.zA, 0, st.mask_words * sizeof(unsigned), c->stream));
        c->mask_scheme = scheme;
    }
    auto enqueue_step = [&] {
        launch(c, KIND_MISC, [&] { k_dt_finalize<<<1, 1, 0, c->stream>>>(c->d_S, cfl, 1); });
        if (scheme == K_MUSCL || scheme == K_MUSCL_MS) {                    // Heun RK2 (A.11)
            run_stage(c, st, st.A, nullptr, st.B, scheme, 0, false);
            run_stage(c, st, st.B, st.A, st.A, scheme, 1, true);
        } else {
            run_stage(c, st, st.A, nullptr, st.A, scheme, 0, true);
        }
    };
    int s0 = 0;
    if (nsteps > 0 && !c->min_valid) {                                       // a9, first step after a state change
        run_dt_reduce(c, st, st.A);
        c->min_valid = true;
    }
    if (c->use_graphs && !c->profile && nsteps >= 2) {
        // capture one step (same kernels, same order, same arguments) and replay it
        if (!c->step_exec || c->graph_scheme != scheme || c->graph_cfl != cfl || c->graph_zoned != c->has_zones ||
            c->graph_masks != c->mk_on) {
            drop_graph(c);
            if (!c->cap_stream) CU(cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking));
            const int64_t l0 = c->launches, h0 = c->halo_bytes;
            cudaStream_t user = c->stream;
            cudaGraph_t graph = nullptr;
            cudaError_t e = cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal);
            if (e == cudaSuccess) {
                c->stream = c->cap_stream;
                enqueue_step();
                c->stream = user;
                e = cudaStreamEndCapture(c->cap_stream, &graph);
            }
            c->graph_launches = c->launches - l0; c->graph_halo = c->halo_bytes - h0;
            c->launches = l0; c->halo_bytes = h0;
            if (e == cudaSuccess) e = cudaGraphInstantiate(&c->step_exec, graph, 0);
            if (graph) cudaGraphDestroy(graph);
            if (e != cudaSuccess) { c->step_exec = nullptr; return fail(SWE_ERR_CUDA, std::string("step graph: ") + cudaGetErrorString(e)); }
            c->graph_scheme = scheme; c->graph_cfl = cfl; c->graph_zoned = c->has_zones; c->graph_masks = c->mk_on;
        }
        for (; s0 < nsteps; ++s0) {
            CU(cudaGraphLaunch(c->step_exec, c->stream));
            c->launches += c->graph_launches; c->halo_bytes += c->graph_halo;
            c->steps++;
        }
    }
    for (int s = s0; s < nsteps; ++s) {
        enqueue_step();
        c->steps++;
    }
    CU(cudaGetLastError());
    c->masks_live = c->mk_on;
    if (c->profile) profile_collect(c);
    if (t_out || last_dt_out) {
        StepScalars hs;
        CU(cudaMemcpyAsync(&hs, c->d_S, sizeof(hs), cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
        if (t_out) *t_out = hs.t;
        if (last_dt_out) *last_dt_out = hs.last_dt;
    }
    return SWE_OK;
}

int swe_fp64_peak(swe_ctx* c, double* tflops_out) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!tflops_out) return fail(SWE_ERR_ARG, "NULL output");
    const int blocks = c->num_sm * 8, iters = 2048;
    double* d = nullptr;
    CU(cudaMalloc((void**)&d, (size_t)blocks * 256 * sizeof(double)));
    cudaEvent_t a, b;
    cudaEventCreate(&a); cudaEventCreate(&b);
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {                 // first repetition warms up
        cudaEventRecord(a, c->stream);
        k_dfma_peak<<<blocks, 256, 0, c->stream>>>(d, iters);
        cudaEventRecord(b, c->stream);
        cudaEventSynchronize(b);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, a, b);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(a); cudaEventDestroy(b);
    cudaFree(d);
    CU(cudaGetLastError());
    *tflops_out = 2.0 * 32.0 * (double)iters * blocks * 256 / (best * 1e-3) / 1e12;
    return SWE_OK;
}

int swe_fastmath_check(swe_ctx* c, int64_t n, const double* a, const double* x, int64_t* ndiff /*2*/, double* maxrel /*2*/) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (n <= 0 || !a || !x || !ndiff || !maxrel) return fail(SWE_ERR_ARG, "bad fastmath_check arguments");
    double *da = nullptr, *dx = nullptr;
    unsigned long long* dout = nullptr;
    const bool dev = is_device_ptr(a) && is_device_ptr(x);
    if (!dev) {
        CU(cudaMalloc((void**)&da, (size_t)n * sizeof(double)));
        cudaError_t e = cudaMalloc((void**)&dx, (size_t)n * sizeof(double));
        if (e != cudaSuccess) { cudaFree(da); return fail(SWE_ERR_CUDA, cudaGetErrorString(e)); }
        cudaMemcpyAsync(da, a, (size_t)n * sizeof(double), cudaMemcpyDefault, c->stream);
        cudaMemcpyAsync(dx, x, (size_t)n * sizeof(double), cudaMemcpyDefault, c->stream);
    }
    cudaError_t e = cudaMalloc((void**)&dout, 4 * sizeof(unsigned long long));
    unsigned long long h[4] = {0, 0, 0, 0};
    if (e == cudaSuccess) {
        cudaMemsetAsync(dout, 0, sizeof(h), c->stream);
        k_fastmath_check<<<grid_for(n, c->grid_light), 256, 0, c->stream>>>(dev ? a : da, dev ? x : dx, (long long)n, dout);
        c->launches++;
        cudaMemcpyAsync(h, dout, sizeof(h), cudaMemcpyDeviceToHost, c->stream);
        e = cudaStreamSynchronize(c->stream);
    }
    cudaFree(da); cudaFree(dx); cudaFree(dout);
    if (e != cudaSuccess) return fail(SWE_ERR_CUDA, cudaGetErrorString(e));
    ndiff[0] = (int64_t)h[0]; ndiff[1] = (int64_t)h[1];
    memcpy(&maxrel[0], &h[2], sizeof(double)); memcpy(&maxrel[1], &h[3], sizeof(double));
    return SWE_OK;
}

int swe_dry_counts(const swe_ctx* cc, int64_t* counts /*5*/) {
    KeepMasks keep_masks(cc);   // read-only
    swe_ctx* c = const_cast<swe_ctx*>(cc);
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!counts) return fail(SWE_ERR_ARG, "NULL output");
    Store& st = c->active();
    unsigned long long* d = nullptr;
    CU(cudaMalloc((void**)&d, 3 * sizeof(unsigned long long)));
    unsigned long long h[3] = {0, 0, 0};
    cudaMemsetAsync(d, 0, sizeof(h), c->stream);
    k_dry_counts<<<grid_for(st.ne, c->grid_light), 256, 0, c->stream>>>(st.dm, st.A, c->P.h_dry, d);
    c->launches++;
    cudaMemcpyAsync(h, d, sizeof(h), cudaMemcpyDeviceToHost, c->stream);
    cudaError_t e = cudaStreamSynchronize(c->stream);
    cudaFree(d);
    if (e != cudaSuccess) return fail(SWE_ERR_CUDA, cudaGetErrorString(e));
    counts[0] = (int64_t)h[0]; counts[1] = (int64_t)h[1]; counts[2] = (int64_t)h[2];
    counts[3] = c->H.nt; counts[4] = c->g.dm.ne_int;
    return SWE_OK;
}

int swe_set_dry_masks(swe_ctx* c, int on) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    c->dry_masks = on != 0;
    return SWE_OK;
}

int swe_set_graphs(swe_ctx* c, int on) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    c->use_graphs = on != 0;
    if (!on) drop_graph(c);
    return SWE_OK;
}

int swe_step_timed(swe_ctx* c, int nsteps, double cfl, int scheme, float* ms_out) {
    const bool live = c && c->masks_live;
    if (check_ctx(c)) return SWE_ERR_ARG;
    c->masks_live = live;               // swe_step with two events around it: nothing else touches the buffers
    cudaEvent_t a, b;
    CU(cudaEventCreate(&a)); CU(cudaEventCreate(&b));
    CU(cudaEventRecord(a, c->stream));
    int rc = swe_step(c, nsteps, cfl, scheme, nullptr, nullptr);
    cudaEventRecord(b, c->stream);
    cudaError_t e = cudaEventSynchronize(b);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, a, b);
    cudaEventDestroy(a); cudaEventDestroy(b);
    if (rc != SWE_OK) return rc;
    if (e != cudaSuccess) return fail(SWE_ERR_CUDA, cudaGetErrorString(e));
    if (ms_out) *ms_out = ms;
    return SWE_OK;
}

int swe_kernel_timed(swe_ctx* c, int which, int scheme, int reps, float* ms_out) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (which < 0 || which > 6 || scheme < 0 || scheme > 3 || reps < 1) return fail(SWE_ERR_ARG, "bad kernel selector");
    Store& st = c->active();
    const bool prof = c->profile; c->profile = false;
    // make the inputs of the timed kernel valid
    if (which >= 2) run_grad(c, st, st.A, scheme);
    if (which >= 3 && which <= 4) run_flux(c, st, st.A, scheme);
    cudaEvent_t a, b;
    CU(cudaEventCreate(&a)); CU(cudaEventCreate(&b));
    CU(cudaEventRecord(a, c->stream));
    for (int r = 0; r < reps; ++r) {
        switch (which) {
            case 0: run_dt_reduce(c, st, st.A); break;
            case 1: run_grad(c, st, st.A, scheme == K_MUSCL_MS ? K_MUSCL_MS : K_MUSCL); break;
            case 2: run_flux(c, st, st.A, scheme); break;
            case 3: run_update(c, st, st.A, nullptr, st.B, 0, false); break;
            case 4: run_update(c, st, st.B, st.A, st.B, 1, false); break;
            case 5: if (c->has_zones) run_exchange_state(c, st.A, 0, c->nsend, true, false); break;
            case 6: if (c->has_zones) run_exchange_state(c, st.A, 0, c->nsend, false, true); break;
        }
    }
    cudaEventRecord(b, c->stream);
    cudaError_t e = cudaEventSynchronize(b);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, a, b);
    cudaEventDestroy(a); cudaEventDestroy(b);
    c->profile = prof;
    if (which == 0) c->min_valid = true;
    if (e != cudaSuccess) return fail(SWE_ERR_CUDA, cudaGetErrorString(e));
    if (ms_out) *ms_out = ms;
    return SWE_OK;
}

int swe_set_profile(swe_ctx* c, int on) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    profile_collect(c);
    c->profile = on != 0;
    for (int k = 0; k < NKIND; ++k) { c->prof_ms[k] = 0.0; c->prof_n[k] = 0; }
    return SWE_OK;
}
int swe_get_profile(swe_ctx* c, double* ms /*7*/, int64_t* count /*7*/) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    profile_collect(c);
    for (int k = 0; k < NKIND; ++k) { if (ms) ms[k] = c->prof_ms[k]; if (count) count[k] = c->prof_n[k]; }
    return SWE_OK;
}

int swe_compute_dt(swe_ctx* c, double cfl, double* dt_out) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!(cfl > 0.0) || !dt_out) return fail(SWE_ERR_ARG, "bad arguments");
    Store& st = c->active();
    run_dt_reduce(c, st, st.A);
    c->min_valid = true;
    StepScalars hs;
    CU(cudaMemcpyAsync(&hs, c->d_S, sizeof(hs), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    double m;
    std::memcpy(&m, &hs.min_bits, sizeof(double));
    *dt_out = std::isinf(m) ? 0.0 : cfl * m;
    return SWE_OK;
}

static int out_to_user(swe_ctx* c, double* out, size_t n, double** dev_out) {
    if (is_device_ptr(out)) { *dev_out = out; return SWE_OK; }
    int rc = ensure_stage(c, n); if (rc) return rc;
    *dev_out = c->d_stage;
    return SWE_OK;
}
static int finish_out(swe_ctx* c, double* out, size_t n, double* dev_out) {
    if (dev_out != out) CU(cudaMemcpyAsync(out, dev_out, n * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return SWE_OK;
}

int swe_gradients(swe_ctx* c, double* out) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!out) return fail(SWE_ERR_ARG, "NULL output");
    if (c->has_zones) return fail(SWE_ERR_STATE, "single-pass inspection calls act on the un-zoned mesh");
    double* d; int rc = out_to_user(c, out, 8 * (size_t)c->g.nc, &d); if (rc) return rc;
    run_grad(c, c->g, c->g.A);
    k_grad_to_user<<<grid_for(c->g.nc, c->grid_light), 256, 0, c->stream>>>(c->g.grad, c->g.d_cell_user, d, (int)c->g.nc);
    CU(cudaGetLastError());
    return finish_out(c, out, 8 * (size_t)c->g.nc, d);
}

int swe_side_fluxes(swe_ctx* c, double dt, int scheme, double* out) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!out || scheme < 0 || scheme > 3) return fail(SWE_ERR_ARG, "bad arguments");
    if (c->has_zones) return fail(SWE_ERR_STATE, "single-pass inspection calls act on the un-zoned mesh");
    double* d; int rc = out_to_user(c, out, 9 * (size_t)c->g.nc, &d); if (rc) return rc;
    k_set_dt<<<1, 1, 0, c->stream>>>(c->d_S, dt);
    run_grad(c, c->g, c->g.A, scheme);
    run_flux(c, c->g, c->g.A, scheme);
    k_side_flux_to_user<<<grid_for(c->g.nc, c->grid_light), 256, 0, c->stream>>>(c->g.dm, c->g.F, c->g.d_cell_user, d);
    CU(cudaGetLastError());
    return finish_out(c, out, 9 * (size_t)c->g.nc, d);
}

int swe_euler_stage(swe_ctx* c, double dt, int scheme, double* h1, double* hu1, double* hv1) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!h1 || !hu1 || !hv1 || scheme < 0 || scheme > 3) return fail(SWE_ERR_ARG, "bad arguments");
    if (c->has_zones) return fail(SWE_ERR_STATE, "single-pass inspection calls act on the un-zoned mesh");
    const int64_t nt = c->g.nc;
    k_set_dt<<<1, 1, 0, c->stream>>>(c->d_S, dt);
    run_grad(c, c->g, c->g.A, scheme);
    run_flux(c, c->g, c->g.A, scheme);
    run_update(c, c->g, c->g.A, nullptr, c->g.B, 0, false);
    const bool dev = is_device_ptr(h1) && is_device_ptr(hu1) && is_device_ptr(hv1);
    double *dh = h1, *dhu = hu1, *dhv = hv1;
    if (!dev) {
        int rc = ensure_stage(c, 3 * (size_t)nt + 2); if (rc) return rc;
        dh = c->d_stage; dhu = c->d_stage + nt; dhv = c->d_stage + 2 * nt;
    }
    k_state_to_user<<<grid_for(nt, c->grid_light), 256, 0, c->stream>>>(c->g.B, c->g.d_cell_user, nullptr, dh, dhu, dhv, (int)nt);
    CU(cudaGetLastError());
    if (!dev) {
        CU(cudaMemcpyAsync(h1, dh, nt * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        CU(cudaMemcpyAsync(hu1, dhu, nt * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        CU(cudaMemcpyAsync(hv1, dhv, nt * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    }
    CU(cudaStreamSynchronize(c->stream));
    return SWE_OK;
}

int swe_get_stats(const swe_ctx* c, int64_t* steps, int64_t* kernel_launches, int64_t* halo_bytes) {
    KeepMasks keep_masks(c);   // read-only
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (steps) *steps = c->steps;
    if (kernel_launches) *kernel_launches = c->launches;
    if (halo_bytes) *halo_bytes = c->halo_bytes;
    return SWE_OK;
}

int swe_account_replays(swe_ctx* c, int64_t steps, int64_t kernel_launches, int64_t halo_bytes) {
    KeepMasks keep_masks(c);
    if (check_ctx(c)) return SWE_ERR_ARG;
    c->steps += steps; c->launches += kernel_launches; c->halo_bytes += halo_bytes;
    return SWE_OK;
}

// ---- zones ----
// Row f4: the ghost layers of all zones on the device (swe_zone_kernels.cuh).  zone_of: per cell of
// the un-zoned mesh, device numbering.  Returns the sorted keys build_zones consumes.
// d_zone: the zone of every cell, already on the device.  keep != nullptr: the sorted keys also stay
// on the device (*keep = their allocation, *d_sorted = the keys; the caller frees *keep).
static bool device_ghost_keys(swe_ctx* c, const int* d_zone, int nz, int nlayers, std::vector<uint64_t>& keys,
                              std::string& err, void** keep = nullptr, unsigned long long** d_sorted = nullptr) {
    const int nc = (int)c->g.nc;
    const int W = (nz + 63) / 64;
    const size_t words = (size_t)W * nc;
    // one arena for the masks (two reach buffers, one fresh buffer per layer) and the two counters;
    // a second one, sized once the number of ghosts is known, for the keys
    unsigned long long *arena = nullptr, *karena = nullptr;
    cudaError_t e = cudaSuccess;
    auto ok = [&](cudaError_t r) { if (e == cudaSuccess) e = r; return e == cudaSuccess; };
    keys.clear();
    if (keep) { *keep = nullptr; *d_sorted = nullptr; }
    const int grid = grid_for(nc, c->grid_light);
    unsigned long long total = 0;
    const size_t nmask = (size_t)(2 + nlayers) * words;
    ok(cudaMalloc((void**)&arena, (nmask + 2) * 8));
    unsigned long long* d_reach[2] = {arena, arena + words};
    unsigned long long* d_fresh[3] = {nullptr, nullptr, nullptr};
    for (int l = 0; l < nlayers; ++l) d_fresh[l] = arena + (size_t)(2 + l) * words;
    unsigned long long* d_count = arena + nmask;             // [0] ghosts found, [1] emit cursor
    if (e == cudaSuccess) {
        ok(cudaMemsetAsync(d_count, 0, 2 * sizeof(unsigned long long), c->stream));
        k_gl_seed<<<grid, 256, 0, c->stream>>>(d_zone, d_reach[0], nc, W);
        for (int l = 0; l < nlayers; ++l)
            k_gl_grow<<<grid, 256, 0, c->stream>>>(c->g.dm.c2c, d_reach[l & 1], d_reach[(l + 1) & 1], d_fresh[l], nc, W, d_count);
        c->launches += 1 + nlayers;
        ok(cudaGetLastError());
        ok(cudaMemcpyAsync(&total, d_count, sizeof(total), cudaMemcpyDeviceToHost, c->stream));
        ok(cudaStreamSynchronize(c->stream));
    }
    if (e == cudaSuccess && total > (unsigned long long)INT32_MAX) { cudaFree(arena); err = "too many ghost cells"; return false; }
    if (e == cudaSuccess && total > 0) {
        const long long n = (long long)total;
        const int nblk = (int)((n + RS_TILE - 1) / RS_TILE);
        if (ok(cudaMalloc((void**)&karena, (size_t)n * 16 + (size_t)256 * nblk * sizeof(unsigned int)))) {
            unsigned long long* d_keys[2] = {karena, karena + n};
            unsigned int* d_hist = (unsigned int*)(karena + 2 * n);
            for (int l = 0; l < nlayers; ++l)
                k_gl_emit<<<grid, 256, 0, c->stream>>>(d_fresh[l], d_zone, l + 1, nz, nc, W, d_keys[0], d_count + 1);
            // significant key bits: 32 (cell) + those of the largest bucket (nz * nz * 4 - 1)
            int bits = 32;
            for (unsigned long long top = (unsigned long long)nz * nz * 4ull - 1ull; top; top >>= 1) ++bits;
            int cur = 0;
            for (int shift = 0; shift < bits; shift += 8) {
                k_rs_hist<<<nblk, RS_THREADS, 0, c->stream>>>(d_keys[cur], n, shift, d_hist, nblk);
                k_rs_scan<<<1, 1024, 0, c->stream>>>(d_hist, (long long)256 * nblk);
                k_rs_scatter<false><<<nblk, RS_THREADS, 0, c->stream>>>(d_keys[cur], d_keys[cur ^ 1], n, shift, d_hist, nblk);
                cur ^= 1;
                c->launches += 3;
            }
            c->launches += nlayers;
            ok(cudaGetLastError());
            keys.resize((size_t)n);
            ok(cudaMemcpyAsync(keys.data(), d_keys[cur], (size_t)n * 8, cudaMemcpyDeviceToHost, c->stream));
            ok(cudaStreamSynchronize(c->stream));
            if (keep && e == cudaSuccess) { *keep = karena; *d_sorted = d_keys[cur]; karena = nullptr; }
        }
    }
    cudaFree(arena); cudaFree(karena);
    if (e != cudaSuccess) { cudaGetLastError(); err = std::string("device ghost-layer generation: ") + cudaGetErrorString(e); return false; }
    return true;
}

// stable LSD radix sort of n 64-bit keys on bits [lo_bit, hi_bit): returns 0 / 1 = the buffer that holds the result
static int rs_sort(swe_ctx* c, unsigned long long* buf[2], long long n, int lo_bit, int hi_bit, unsigned int* d_hist,
                   unsigned int* val[2] = nullptr) {
    const int nblk = (int)((n + RS_TILE - 1) / RS_TILE);
    int cur = 0;
    for (int shift = lo_bit; shift < hi_bit; shift += 8) {
        k_rs_hist<<<nblk, RS_THREADS, 0, c->stream>>>(buf[cur], n, shift, d_hist, nblk);
        k_rs_scan<<<1, 1024, 0, c->stream>>>(d_hist, (long long)256 * nblk);
        if (val) k_rs_scatter<true><<<nblk, RS_THREADS, 0, c->stream>>>(buf[cur], buf[cur ^ 1], n, shift, d_hist, nblk, val[cur], val[cur ^ 1]);
        else k_rs_scatter<false><<<nblk, RS_THREADS, 0, c->stream>>>(buf[cur], buf[cur ^ 1], n, shift, d_hist, nblk);
        cur ^= 1;
        c->launches += 3;
    }
    return cur;
}
static int bits_of(unsigned long long v) { int b = 0; for (; v; v >>= 1) ++b; return b; }

// A.12.1 on the device (swe_zone_assembly.cuh): d_zone[cell] = zone of every cell, nz a power of two
static int device_rcb(swe_ctx* c, int nz, int* d_zone) {
    const int nc = (int)c->g.nc;
    const int grid = grid_for(nc, c->grid_light);
    if (nz == 1) { CU(cudaMemsetAsync(d_zone, 0, (size_t)nc * sizeof(int), c->stream)); return SWE_OK; }
    Scratch tmp;
    unsigned long long* k[2][2] = {{nullptr, nullptr}, {nullptr, nullptr}};     // [axis][ping-pong]
    unsigned int* v[2] = {nullptr, nullptr};
    unsigned int* d_hist = nullptr;
    int* d_user_cell = nullptr;
    long long* d_seg = nullptr;
    double* d_c[2] = {nullptr, nullptr};
    for (int a = 0; a < 2; ++a) for (int b = 0; b < 2; ++b) CU(tmp.get(&k[a][b], (size_t)nc));
    CU(tmp.get(&v[0], (size_t)nc)); CU(tmp.get(&v[1], (size_t)nc));
    CU(tmp.get(&d_hist, (size_t)256 * (size_t)((nc + RS_TILE - 1) / RS_TILE)));
    CU(tmp.get(&d_user_cell, (size_t)nc)); CU(tmp.get(&d_seg, (size_t)nz + 1)); CU(tmp.get(&d_c[0], (size_t)nc)); CU(tmp.get(&d_c[1], (size_t)nc));
    CU(cudaMemcpyAsync(d_user_cell, c->H.user_cell.data(), (size_t)nc * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    CU(cudaMemcpyAsync(d_c[0], c->H.cx.data(), (size_t)nc * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    CU(cudaMemcpyAsync(d_c[1], c->H.cy.data(), (size_t)nc * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    int cur[2] = {0, 0};
    for (int a = 0; a < 2; ++a) {                    // the two global orders
        k_rcb_init<<<grid, 256, 0, c->stream>>>(d_user_cell, d_c[a], k[a][0], v[0], nc);
        const int r = rs_sort(c, k[a], nc, 0, 64, d_hist, v);
        k_rcb_order<<<grid, 256, 0, c->stream>>>(v[r], k[a][0], nc);
        cur[a] = 0;
    }
    std::vector<long long> seg{0, nc};
    int levels = 0;
    for (int m = nz; m > 1; m >>= 1) ++levels;
    for (int l = 0; l < levels; ++l) {
        const int nseg = (int)seg.size() - 1;
        CU(cudaMemcpyAsync(d_seg, seg.data(), seg.size() * sizeof(long long), cudaMemcpyHostToDevice, c->stream));
        k_rcb_mark<<<grid, 256, 0, c->stream>>>(k[0][cur[0]], k[1][cur[1]], d_c[0], d_c[1], d_seg, nseg, d_zone, nc);
        for (int a = 0; a < 2; ++a) {
            k_rcb_rekey<<<grid, 256, 0, c->stream>>>(k[a][cur[a]], d_zone, nc);
            unsigned long long* pp[2] = {k[a][cur[a]], k[a][cur[a] ^ 1]};
            const int r = rs_sort(c, pp, nc, 32, 32 + l + 1, d_hist);
            cur[a] ^= r;
        }
        CU(cudaStreamSynchronize(c->stream));          // seg is re-uploaded next level
        std::vector<long long> nxt;
        for (int s2 = 0; s2 < nseg; ++s2) { nxt.push_back(seg[s2]); nxt.push_back(seg[s2] + (seg[s2 + 1] - seg[s2]) / 2); }
        nxt.push_back(nc);
        seg.swap(nxt);
        c->launches += 3;
    }
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(c->stream));
    return SWE_OK;
}

static int zones_create_impl(swe_ctx* c, int nzones, int nlayers, const int32_t* zone_of_cell, int nranks,
                             int rank, const int32_t* zone_begin) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (nzones < 0) return fail(SWE_ERR_ARG, "nzones must be >= 0");
    int rc = sync_global_from_zoned(c); if (rc) return rc;
    CU(cudaStreamSynchronize(c->stream));
    free_zones(c);
    c->min_valid = false;
    k_reset_min<<<1, 1, 0, c->stream>>>(c->d_S);
    if (nzones == 0) return SWE_OK;
    std::vector<int32_t> hz;
    if (zone_of_cell && is_device_ptr(zone_of_cell)) {
        hz.resize(c->H.nt);
        CU(cudaMemcpy(hz.data(), zone_of_cell, c->H.nt * sizeof(int32_t), cudaMemcpyDeviceToHost));
        zone_of_cell = hz.data();
    }
    std::string err;
    bool ok = false;
    const auto t0 = std::chrono::steady_clock::now();
    auto ms_since = [&](std::chrono::steady_clock::time_point a) {
        return std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - a).count(); };
    Scratch tmp;
    const bool trace = getenv("SWE_ZONE_TRACE") != nullptr;
    auto mark = [&](const char* what) {
        if (!trace) return;
        cudaStreamSynchronize(c->stream);
        fprintf(stderr, "[swe zones] %-28s %8.1f ms\n", what, ms_since(t0));
    };
    const int nc = (int)c->g.nc;
    const int nz = nzones;
    if (nlayers < 1 || nlayers > 3) return fail(SWE_ERR_ARG, "nlayers must be 1, 2 or 3");
    if ((int64_t)nz * nz > (int64_t)1 << 29) return fail(SWE_ERR_ARG, "too many zones");
    const int grid = grid_for(nc, c->grid_light);

    // ---- A.12.1 the zone of every cell (device numbering) ----
    ZoneDeviceLists dev;
    if (zone_of_cell) {
        dev.zone_of.resize(nc);
        for (int i = 0; i < nc; ++i) {
            const int32_t zc = zone_of_cell[c->H.m.cell_user[i]];
            if (zc < 0 || zc >= nz) return fail(SWE_ERR_ARG, "zone_of_cell value out of range");
            dev.zone_of[i] = zc;
        }
    }
    int* d_zone = nullptr;
    CU(tmp.get(&d_zone, (size_t)nc));
    if (zone_of_cell) {
        CU(cudaMemcpyAsync(d_zone, dev.zone_of.data(), (size_t)nc * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    } else {
        if (nz & (nz - 1)) return fail(SWE_ERR_ARG, "recursive coordinate bisection needs a power-of-two nzones");
        rc = device_rcb(c, nz, d_zone); if (rc) return rc;       // the zone ids stay on the device
    }
    c->zone_ms[3] = ms_since(t0);

    mark("zone of every cell");
    // ---- A.12.2-3 ghost layers of all zones: sorted keys, on the host and still on the device ----
    std::vector<uint64_t> hkeys;
    void* keep = nullptr; unsigned long long* d_gkeys = nullptr;
    const auto g0 = std::chrono::steady_clock::now();
    if (!device_ghost_keys(c, d_zone, nz, nlayers, hkeys, err, &keep, &d_gkeys)) return fail(SWE_ERR_CUDA, err);
    if (keep) tmp.p.push_back(keep);
    c->zone_ms[0] = ms_since(g0);
    const long long nk = (long long)hkeys.size();

    mark("ghost layers");
    // ---- owned cells: one stable radix pass per 8 zone bits over (zone << 32 | cell) ----
    unsigned long long* okeys[2] = {nullptr, nullptr};
    unsigned int* d_hist = nullptr;
    long long* d_start = nullptr;
    int *d_opos = nullptr, *d_kopos = nullptr;
    CU(tmp.get(&okeys[0], (size_t)nc)); CU(tmp.get(&okeys[1], (size_t)nc));
    CU(tmp.get(&d_start, (size_t)nz + 1));
    CU(tmp.get(&d_opos, (size_t)nc));
    CU(tmp.get(&d_kopos, (size_t)nk));
    const long long ne_int_g = c->g.dm.ne_int;
    {
        const long long nmax = std::max<long long>(std::max<long long>(nc, 2 * ne_int_g), 1);
        CU(tmp.get(&d_hist, (size_t)256 * (size_t)((nmax + RS_TILE - 1) / RS_TILE)));
    }
    k_za_owned_keys<<<grid, 256, 0, c->stream>>>(d_zone, okeys[0], nc);
    const int ocur = rs_sort(c, okeys, nc, 32, 32 + bits_of((unsigned long long)nz - 1), d_hist);
    CU(cudaMemsetAsync(d_start, 0xff, ((size_t)nz + 1) * sizeof(long long), c->stream));
    k_za_starts<<<grid, 256, 0, c->stream>>>(okeys[ocur], nc, d_start);
    std::vector<long long> ostart((size_t)nz + 1);
    CU(cudaMemcpyAsync(ostart.data(), d_start, ((size_t)nz + 1) * sizeof(long long), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    ostart[nz] = nc;
    for (int z = nz - 1; z >= 0; --z) if (ostart[z] < 0) ostart[z] = ostart[z + 1];       // zones without cells
    CU(cudaMemcpyAsync(d_start, ostart.data(), ((size_t)nz + 1) * sizeof(long long), cudaMemcpyHostToDevice, c->stream));
    k_za_owned_pos<<<grid, 256, 0, c->stream>>>(okeys[ocur], d_start, d_opos, nc);
    dev.nowned.resize(nz);
    for (int z = 0; z < nz; ++z) dev.nowned[z] = ostart[z + 1] - ostart[z];
    dev.key_owned_pos.resize((size_t)nk);
    if (nk) {
        k_za_key_opos<<<grid_for(nk, c->grid_light), 256, 0, c->stream>>>(d_gkeys, nk, d_opos, d_kopos);
        CU(cudaMemcpyAsync(dev.key_owned_pos.data(), d_kopos, (size_t)nk * sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    }
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(c->stream));
    c->launches += 4;

    mark("owned positions");
    // ---- links, send lists, exchange lists per rank: the host, from the keys (O(ghost cells)) ----
    GhostFinder finder = [&](const std::vector<int32_t>&, int, int, std::vector<uint64_t>& keys, std::string&) {
        keys = hkeys; return true; };
    try { ok = build_zones(c->H, c->Z, nz, nlayers, nullptr, err, nranks, rank, zone_begin, finder, &dev, false); }
    catch (const std::bad_alloc&) { c->Z = ZoneSet(); return fail(SWE_ERR_NOMEM, "out of host memory in zone set-up"); }
    if (!ok) { c->Z = ZoneSet(); return fail(SWE_ERR_ARG, err); }
    c->zone_ms[1] = ms_since(t0);

    mark("host lists");
    // ---- the concatenated zoned mesh, assembled on the device (swe_zone_assembly.cuh) ----
    std::vector<int> zres(nz, -1), zid;
    std::vector<long long> coff, nown, ownstart, ghstart, ghend;
    {
        size_t kp = 0;
        for (int z = 0; z < nz; ++z) {
            const size_t k0 = kp;
            while (kp < hkeys.size() && (int64_t)(((hkeys[kp] >> 32) >> 2) / (uint64_t)nz) == z) ++kp;
            if (c->Z.zone_rank[z] != rank) continue;
            zres[z] = (int)zid.size(); zid.push_back(z);
            coff.push_back(c->Z.z[z].offset); nown.push_back(c->Z.z[z].nowned); ownstart.push_back(ostart[z]);
            ghstart.push_back((long long)k0); ghend.push_back((long long)kp);
        }
    }
    const int nzr = (int)zid.size();
    long long ncz = 0;
    for (int r = 0; r < nzr; ++r) ncz = std::max(ncz, coff[r] + c->Z.z[zid[r]].ncells);
    coff.push_back(ncz);
    if (nzr == 0 || ncz == 0) return fail(SWE_ERR_ARG, "this rank holds no zone");
    ZoneTabs T{};
    T.nz = nz; T.nzr = nzr; T.nlayers = nlayers; T.gl = (nlayers >= 2) ? 1 : 0;
    int *d_zres = nullptr, *d_zid = nullptr;
    long long* d_tab = nullptr;                      // coff | nown | ownstart | ghstart | ghend | ioff | boff
    const size_t TS = (size_t)nzr + 1;
    CU(tmp.get(&d_zres, (size_t)nz)); CU(tmp.get(&d_zid, (size_t)nzr)); CU(tmp.get(&d_tab, 7 * TS));
    CU(cudaMemcpyAsync(d_zres, zres.data(), (size_t)nz * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    CU(cudaMemcpyAsync(d_zid, zid.data(), (size_t)nzr * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    auto put_tab = [&](int slot, const std::vector<long long>& v) {
        return cudaMemcpyAsync(d_tab + slot * TS, v.data(), v.size() * sizeof(long long), cudaMemcpyHostToDevice, c->stream); };
    CU(put_tab(0, coff)); CU(put_tab(1, nown)); CU(put_tab(2, ownstart)); CU(put_tab(3, ghstart)); CU(put_tab(4, ghend));
    T.zres = d_zres; T.zid = d_zid; T.coff = d_tab; T.nown = d_tab + TS; T.ownstart = d_tab + 2 * TS;
    T.ghstart = d_tab + 3 * TS; T.ghend = d_tab + 4 * TS; T.ioff = d_tab + 5 * TS; T.boff = d_tab + 6 * TS;

    Store& st = c->z;
    st.nc = ncz;
    int* d_src = nullptr; uint8_t* d_lay = nullptr;
    CU(cudaMalloc((void**)&c->d_src_of_cell, (size_t)ncz * sizeof(int)));
    d_src = c->d_src_of_cell;
    CU(st.alloc(&d_lay, (size_t)ncz));
    const int gridz = grid_for(ncz, c->grid_light);
    k_za_cells<<<gridz, 256, 0, c->stream>>>(T, okeys[ocur], d_gkeys, d_src, d_lay, (int)ncz);

    mark("cells");
    // edges: count, emit, sort by (zone, global edge)
    unsigned long long* d_cnt = nullptr;
    CU(tmp.get(&d_cnt, 4));
    CU(cudaMemsetAsync(d_cnt, 0, 4 * sizeof(unsigned long long), c->stream));
    k_za_int_edges<<<grid_for(ne_int_g, c->grid_light), 256, 0, c->stream>>>(T, d_zone, c->g.dm.elr, (int)ne_int_g, nullptr, d_cnt);
    k_za_bnd_edges<<<gridz, 256, 0, c->stream>>>(T, d_src, d_lay, c->g.dm.c2c, (int)ncz, nullptr, d_cnt + 1);
    unsigned long long cnt[2] = {0, 0};
    CU(cudaMemcpyAsync(cnt, d_cnt, sizeof(cnt), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    const long long ni = (long long)cnt[0], nb = (long long)cnt[1];
    if (ni + nb > (long long)INT32_MAX / 2) return fail(SWE_ERR_ARG, "zoned mesh too large");
    unsigned long long *ikeys[2] = {nullptr, nullptr}, *bkeys[2] = {nullptr, nullptr};
    CU(tmp.get(&ikeys[0], (size_t)ni)); CU(tmp.get(&ikeys[1], (size_t)ni));
    CU(tmp.get(&bkeys[0], (size_t)nb)); CU(tmp.get(&bkeys[1], (size_t)nb));
    k_za_int_edges<<<grid_for(ne_int_g, c->grid_light), 256, 0, c->stream>>>(T, d_zone, c->g.dm.elr, (int)ne_int_g, ikeys[0], d_cnt + 2);
    k_za_bnd_edges<<<gridz, 256, 0, c->stream>>>(T, d_src, d_lay, c->g.dm.c2c, (int)ncz, bkeys[0], d_cnt + 3);
    const int kbits = 32 + bits_of((unsigned long long)nzr - 1);
    const int icur = ni ? rs_sort(c, ikeys, ni, 0, kbits, d_hist) : 0;
    const int bcur = nb ? rs_sort(c, bkeys, nb, 0, kbits, d_hist) : 0;
    mark("edge keys sorted");
    // per-zone ranges of the two sorted edge lists
    std::vector<long long> ioff(TS), boff(TS);
    {
        long long* d_es = nullptr;
        CU(tmp.get(&d_es, 2 * TS));
        CU(cudaMemsetAsync(d_es, 0xff, 2 * TS * sizeof(long long), c->stream));
        if (ni) k_za_starts<<<grid_for(ni, c->grid_light), 256, 0, c->stream>>>(ikeys[icur], ni, d_es);
        if (nb) k_za_starts<<<grid_for(nb, c->grid_light), 256, 0, c->stream>>>(bkeys[bcur], nb, d_es + TS);
        CU(cudaMemcpyAsync(ioff.data(), d_es, TS * sizeof(long long), cudaMemcpyDeviceToHost, c->stream));
        CU(cudaMemcpyAsync(boff.data(), d_es + TS, TS * sizeof(long long), cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
        ioff[nzr] = ni; boff[nzr] = nb;
        for (int r = nzr - 1; r >= 0; --r) { if (ioff[r] < 0) ioff[r] = ioff[r + 1]; if (boff[r] < 0) boff[r] = boff[r + 1]; }
        for (size_t r = 0; r < TS; ++r) boff[r] += ni;                  // boundary edges follow all interior edges
        CU(put_tab(5, ioff)); CU(put_tab(6, boff));
    }
    const long long nez = ni + nb;
    st.ne = nez; st.nbe = nb;
    DevMesh& d = st.dm;
    d = DevMesh{};
    d.nc = (int)ncz; d.ne = (int)nez; d.ne_int = (int)ni; d.glayer = T.gl;
    ZoneCellOut CO{}; ZoneEdgeOut EO{};
    CU(st.alloc(&CO.c2c, (size_t)ncz)); CU(st.alloc(&CO.c2e, (size_t)ncz)); CU(st.alloc(&CO.cell_user, (size_t)ncz));
    CU(st.alloc(&CO.zc, (size_t)ncz)); CU(st.alloc(&CO.area, (size_t)ncz)); CU(st.alloc(&CO.rin, (size_t)ncz));
    CU(st.alloc(&CO.dupw, (size_t)ncz));
    for (int k = 0; k < 3; ++k) CU(st.alloc(&CO.w[k], (size_t)ncz));
    CU(st.alloc(&CO.r[0], (size_t)ncz)); CU(st.alloc(&CO.r[1], (size_t)ncz)); CU(st.alloc(&CO.rres, (size_t)ncz));
    CU(st.alloc(&EO.elr, (size_t)nez)); CU(st.alloc(&EO.en, (size_t)nez)); CU(st.alloc(&EO.elen, (size_t)nez));
    CU(st.alloc(&EO.edx, (size_t)nez)); CU(st.alloc(&EO.erl, (size_t)nez)); CU(st.alloc(&EO.err, (size_t)nez));
    CU(st.alloc(&EO.edlr, (size_t)nez)); CU(st.alloc(&EO.ernorm, (size_t)nez)); CU(st.alloc(&EO.eside, (size_t)nez));
    CU(st.alloc(&EO.ed, (size_t)nez));
    int* d_gedge = nullptr;
    CU(tmp.get(&d_gedge, (size_t)nb));
    EO.gedge = d_gedge;
    k_za_fill_cells<<<gridz, 256, 0, c->stream>>>(T, c->g.dm, c->g.d_cell_user, d_zone, d_opos, d_gkeys, ikeys[icur], bkeys[bcur],
                                                  d_src, d_lay, CO, (int)ncz, ni);
    k_za_fill_edges<<<grid_for(nez, c->grid_light), 256, 0, c->stream>>>(T, c->g.dm, d_zone, d_opos, d_gkeys, ikeys[icur], bkeys[bcur],
                                                                         EO, ni, nez);
    c->launches += 7;
    CU(cudaGetLastError());
    d.c2c = CO.c2c; d.c2e = CO.c2e; d.zc = CO.zc; d.area = CO.area; d.rin = CO.rin; d.dupw = CO.dupw;
    for (int k = 0; k < 3; ++k) d.w[k] = CO.w[k];
    d.r[0] = CO.r[0]; d.r[1] = CO.r[1]; d.r[2] = nullptr; d.rres = CO.rres;
    d.nman_tab = c->d_nman_tab;
    st.d_c2e = CO.c2e;
    d.elr = EO.elr; d.en = EO.en; d.elen = EO.elen; d.edx = EO.edx; d.erl = EO.erl; d.err = EO.err;
    d.edlr = EO.edlr; d.ernorm = EO.ernorm; d.eside = EO.eside; d.ed = EO.ed;
    d.layer = d_lay;
    st.d_cell_user = CO.cell_user;
    mark("arrays filled");
    // cells on a send list carry -1 in c2e.w (overlap schedule)
    c->nsendcells = (int64_t)c->Z.send_cells.size();
    CU(cudaMalloc((void**)&c->d_send_cells, (size_t)(c->nsendcells ? c->nsendcells : 1) * sizeof(int)));
    if (c->nsendcells) {
        CU(cudaMemcpyAsync(c->d_send_cells, c->Z.send_cells.data(), c->nsendcells * sizeof(int), cudaMemcpyHostToDevice, c->stream));
        k_za_mark_send<<<grid_for(c->nsendcells, c->grid_light), 256, 0, c->stream>>>(CO.c2e, c->d_send_cells, (int)c->nsendcells);
    }
    // boundary kinds / values follow the tags of the global edges; state, gradient and flux buffers
    {
        std::vector<int> ge((size_t)nb);
        if (nb) CU(cudaMemcpyAsync(ge.data(), d_gedge, (size_t)nb * sizeof(int), cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
        st.h_btag.assign((size_t)nb, -1);
        for (long long j = 0; j < nb; ++j) st.h_btag[j] = c->g.h_btag[ge[j] - ne_int_g];
    }
    CU(st.alloc(&st.d_bkind, (size_t)nb)); CU(st.alloc(&st.d_bval, (size_t)nb)); CU(st.alloc(&st.d_nman, (size_t)ncz));
    d.bkind = st.d_bkind; d.bval = st.d_bval; d.nman = st.d_nman;
    CU(st.alloc(&st.A, (size_t)ncz)); CU(st.alloc(&st.B, (size_t)ncz)); CU(st.alloc(&st.grad, 3 * (size_t)ncz));
    CU(st.alloc(&st.F.f1, (size_t)nez)); CU(st.alloc(&st.F.fxl, (size_t)nez)); CU(st.alloc(&st.F.fyl, (size_t)nez));
    CU(st.alloc(&st.F.fxr, (size_t)nez)); CU(st.alloc(&st.F.fyr, (size_t)nez));
    {
        const size_t wc = ((size_t)ncz + 31) / 32 + 1, we = ((size_t)nez + 31) / 32 + 1;
        st.mask_words = 3 * wc + we;
        CU(st.alloc(&st.zA, st.mask_words));
        st.zB = st.zA + wc; st.gz = st.zB + wc; st.fz = st.gz + wc;
    }
    CU(cudaMemsetAsync(st.grad, 0, 3 * (size_t)ncz * sizeof(double4), c->stream));
    mark("buffers allocated");
    // the host's copy of the cell lists is fetched when swe_zone_cells asks for it (zone_cells_to_host)
    c->zr_zone = zid; c->zr_off = coff;
    c->zone_ms[4] = ms_since(t0);
    c->nsend = (int64_t)c->Z.send_idx.size();
    const size_t ns = (size_t)(c->nsend ? c->nsend : 1);
    CU(cudaMalloc((void**)&c->d_send_idx, ns * sizeof(int)));
    CU(cudaMalloc((void**)&c->d_recv_idx, ns * sizeof(int)));
    CU(cudaMalloc((void**)&c->d_sendbuf, ns * 8 * sizeof(double)));
    if (c->nsend) {
        CU(cudaMemcpyAsync(c->d_send_idx, c->Z.send_idx.data(), c->nsend * sizeof(int), cudaMemcpyHostToDevice, c->stream));
        CU(cudaMemcpyAsync(c->d_recv_idx, c->Z.recv_idx.data(), c->nsend * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    }
    c->nrsend = (int64_t)c->Z.rsend_idx.size();
    c->nrrecv = (int64_t)c->Z.rrecv_idx.size();
    CU(cudaMalloc((void**)&c->d_rsend_idx, (size_t)(c->nrsend ? c->nrsend : 1) * sizeof(int)));
    CU(cudaMalloc((void**)&c->d_rrecv_idx, (size_t)(c->nrrecv ? c->nrrecv : 1) * sizeof(int)));
    if (c->nrsend) CU(cudaMemcpyAsync(c->d_rsend_idx, c->Z.rsend_idx.data(), c->nrsend * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    if (c->nrrecv) CU(cudaMemcpyAsync(c->d_rrecv_idx, c->Z.rrecv_idx.data(), c->nrrecv * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    CU(cudaMalloc((void**)&c->d_rsend_dst, (size_t)(c->nrsend ? c->nrsend : 1) * sizeof(int)));
    CU(cudaMalloc((void**)&c->d_rsend_peer, (size_t)(c->nrsend ? c->nrsend : 1) * sizeof(int)));
    if (c->nrsend) {
        CU(cudaMemcpyAsync(c->d_rsend_dst, c->Z.rsend_dst.data(), c->nrsend * sizeof(int), cudaMemcpyHostToDevice, c->stream));
        CU(cudaMemcpyAsync(c->d_rsend_peer, c->Z.rsend_peer.data(), c->nrsend * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    }
    CU(cudaMalloc((void**)&c->d_peerA, (size_t)nranks * sizeof(double4*)));
    CU(cudaMalloc((void**)&c->d_peerB, (size_t)nranks * sizeof(double4*)));
    c->peerA.assign(nranks, nullptr); c->peerB.assign(nranks, nullptr); c->peer_ipc.assign(nranks, 0);
    c->peerA[rank] = c->z.A; c->peerB[rank] = c->z.B;
    c->has_zones = true;
    rc = refresh_bc(c, c->z); if (rc) return rc;
    k_gather_cells<<<grid_for(c->z.nc, c->grid_light), 256, 0, c->stream>>>(c->z.A, c->g.A, c->d_src_of_cell, (int)c->z.nc);
    k_gather_cells<<<grid_for(c->z.nc, c->grid_light), 256, 0, c->stream>>>(c->z.B, c->g.A, c->d_src_of_cell, (int)c->z.nc);
    k_gather_scalar<<<grid_for(c->z.nc, c->grid_light), 256, 0, c->stream>>>(c->z.d_nman, c->g.d_nman, c->d_src_of_cell, (int)c->z.nc);
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(c->stream));
    c->zone_ms[2] = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
    return SWE_OK;
}

int swe_zones_create(swe_ctx* c, int nzones, int nlayers, const int32_t* zone_of_cell) {
    return zones_create_impl(c, nzones, nlayers, zone_of_cell, 1, 0, nullptr);
}

// ---- zones distributed over ranks (scope row f3): the caller moves the halo buffers ----
int swe_zones_create_dist(swe_ctx* c, int nzones, int nlayers, const int32_t* zone_of_cell, int nranks,
                          int rank, const int32_t* zone_begin) {
    if (nzones < 1 || nranks < 1 || rank < 0 || rank >= nranks || (nranks > 1 && !zone_begin))
        return fail(SWE_ERR_ARG, "bad distributed zone arguments");
    return zones_create_impl(c, nzones, nlayers, zone_of_cell, nranks, rank, zone_begin);
}

int swe_halo_counts(const swe_ctx* c, int64_t* send_cells, int64_t* recv_cells) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!c->has_zones) return fail(SWE_ERR_STATE, "no zones");
    for (int p = 0; p < c->Z.nranks; ++p) {
        if (send_cells) send_cells[p] = c->Z.rsend_off[p + 1] - c->Z.rsend_off[p];
        if (recv_cells) recv_cells[p] = c->Z.rrecv_off[p + 1] - c->Z.rrecv_off[p];
    }
    return SWE_OK;
}

int swe_halo_pack(swe_ctx* c, int buffer, double* sendbuf) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!c->has_zones) return fail(SWE_ERR_STATE, "no zones");
    if (buffer < 0 || buffer > 1 || (c->nrsend && (!sendbuf || !is_device_ptr(sendbuf)))) return fail(SWE_ERR_ARG, "bad halo buffer");
    if (c->nrsend) {
        launch(c, KIND_PACK, [&] {
            k_pack_state<<<grid_for(c->nrsend, c->grid_light), 256, 0, c->stream>>>(buffer ? c->z.B : c->z.A, c->d_rsend_idx, sendbuf, 0, c->nrsend);
        });
        c->halo_bytes += c->nrsend * (4 + 32 + 24);
    }
    CU(cudaGetLastError());
    return SWE_OK;
}

int swe_halo_unpack(swe_ctx* c, int buffer, const double* recvbuf) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!c->has_zones) return fail(SWE_ERR_STATE, "no zones");
    if (buffer < 0 || buffer > 1 || (c->nrrecv && (!recvbuf || !is_device_ptr(recvbuf)))) return fail(SWE_ERR_ARG, "bad halo buffer");
    if (c->nrrecv) {
        launch(c, KIND_UNPACK, [&] {
            k_unpack_state<<<grid_for(c->nrrecv, c->grid_light), 256, 0, c->stream>>>(buffer ? c->z.B : c->z.A, c->d_rrecv_idx, recvbuf, c->z.dm.zc, 0, c->nrrecv);
        });
        c->halo_bytes += c->nrrecv * (4 + 24 + 8 + 32);
    }
    run_exchange_state(c, buffer ? c->z.B : c->z.A, 0, c->nsend, true, true);    // links between resident zones
    CU(cudaGetLastError());
    return SWE_OK;
}

// ---- halo exchange as one kernel over peer memory ----
static int peer_store(swe_ctx* c, int peer, void* A, void* B, bool ipc) {
    cudaError_t e = cudaSuccess;
    if (c->peer_ipc[peer]) {
        cudaStreamSynchronize(c->stream);                 // no push through the old mapping is still running
        e = cudaIpcCloseMemHandle(c->peerA[peer]);
        const cudaError_t e2 = cudaIpcCloseMemHandle(c->peerB[peer]);
        if (e == cudaSuccess) e = e2;
    }
    c->peerA[peer] = A; c->peerB[peer] = B; c->peer_ipc[peer] = ipc ? 1 : 0;
    if (e != cudaSuccess) { cudaGetLastError(); return fail(SWE_ERR_CUDA, std::string("cudaIpcCloseMemHandle: ") + cudaGetErrorString(e)); }
    return SWE_OK;
}
static int peer_upload(swe_ctx* c) {
    const size_t n = c->peerA.size();
    CU(cudaMemcpyAsync(c->d_peerA, c->peerA.data(), n * sizeof(void*), cudaMemcpyHostToDevice, c->stream));
    CU(cudaMemcpyAsync(c->d_peerB, c->peerB.data(), n * sizeof(void*), cudaMemcpyHostToDevice, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return SWE_OK;
}
static int check_peer(swe_ctx* c, int peer) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!c->has_zones) return fail(SWE_ERR_STATE, "no zones");
    if (peer < 0 || peer >= c->Z.nranks || peer == c->Z.rank) return fail(SWE_ERR_ARG, "peer must be another rank");
    return SWE_OK;
}

int swe_peer_export(swe_ctx* c, unsigned char* handles) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!c->has_zones) return fail(SWE_ERR_STATE, "no zones");
    if (!handles) return fail(SWE_ERR_ARG, "NULL handle buffer");
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "IPC handle size");
    cudaIpcMemHandle_t h;
    CU(cudaIpcGetMemHandle(&h, c->z.A));
    std::memcpy(handles, &h, 64);
    CU(cudaIpcGetMemHandle(&h, c->z.B));
    std::memcpy(handles + 64, &h, 64);
    return SWE_OK;
}

int swe_peer_import(swe_ctx* c, int peer, const unsigned char* handles) {
    int rc = check_peer(c, peer); if (rc) return rc;
    if (!handles) return fail(SWE_ERR_ARG, "NULL handle buffer");
    // whatever was mapped for this peer goes first: opening a handle that is already open in this
    // process is an error on some CUDA versions (re-import after a transport fallback, tests)
    rc = peer_store(c, peer, nullptr, nullptr, false);
    cudaIpcMemHandle_t h;
    void *A = nullptr, *B = nullptr;
    std::memcpy(&h, handles, 64);
    cudaError_t e = cudaIpcOpenMemHandle(&A, h, cudaIpcMemLazyEnablePeerAccess);
    if (e == cudaSuccess) {
        std::memcpy(&h, handles + 64, 64);
        e = cudaIpcOpenMemHandle(&B, h, cudaIpcMemLazyEnablePeerAccess);
        if (e != cudaSuccess) { cudaIpcCloseMemHandle(A); A = nullptr; }
    }
    if (e != cudaSuccess) {
        cudaGetLastError();
        peer_upload(c);      // the peer's slots are NULL again on the device too: swe_halo_push refuses instead of pushing through stale pointers
        return fail(SWE_ERR_CUDA, std::string("cudaIpcOpenMemHandle: ") + cudaGetErrorString(e));
    }
    if (rc == SWE_OK) rc = peer_store(c, peer, A, B, true);
    if (rc != SWE_OK) return rc;
    return peer_upload(c);
}

int swe_peer_raw(swe_ctx* c, void** A, void** B) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!c->has_zones) return fail(SWE_ERR_STATE, "no zones");
    if (A) *A = c->z.A;
    if (B) *B = c->z.B;
    return SWE_OK;
}

int swe_peer_set_raw(swe_ctx* c, int peer, void* A, void* B) {
    int rc = check_peer(c, peer); if (rc) return rc;
    if (!A || !B || !is_device_ptr(A) || !is_device_ptr(B)) return fail(SWE_ERR_ARG, "peer buffers must be device pointers");
    rc = peer_store(c, peer, A, B, false);
    if (rc != SWE_OK) { peer_upload(c); return rc; }
    return peer_upload(c);
}

int swe_halo_push(swe_ctx* c, int buffer) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!c->has_zones) return fail(SWE_ERR_STATE, "no zones");
    if (buffer < 0 || buffer > 1) return fail(SWE_ERR_ARG, "bad halo buffer");
    for (int p = 0; p < c->Z.nranks; ++p)
        if (c->Z.rsend_off[p + 1] > c->Z.rsend_off[p] && !c->peerA[p])
            return fail(SWE_ERR_STATE, "swe_halo_push: a peer this rank sends to has not been imported");
    double4* U = buffer ? c->z.B : c->z.A;
    if (c->nrsend) {
        launch(c, KIND_PACK, [&] {
            k_halo_push<<<grid_for(c->nrsend, c->grid_light * 4, 64), 64, 0, c->stream>>>(U, c->d_rsend_idx, c->d_rsend_dst, c->d_rsend_peer,
                                                                                  buffer ? c->d_peerB : c->d_peerA, c->nrsend);
        });
        c->halo_bytes += c->nrsend * (12 + 32 + 32);
    }
    run_exchange_state(c, U, 0, c->nsend, true, true);    // links between resident zones
    CU(cudaGetLastError());
    return SWE_OK;
}

int swe_dist_local_min(swe_ctx* c, double* min_out) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!min_out || !is_device_ptr(min_out)) return fail(SWE_ERR_ARG, "min_out must be a device pointer");
    Store& st = c->active();
    if (!c->min_valid) run_dt_reduce(c, st, st.A);
    c->min_valid = true;
    CU(cudaMemcpyAsync(min_out, &c->d_S->min_bits, sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
    return SWE_OK;
}

int swe_dist_begin_step(swe_ctx* c, const double* min_in, double cfl) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!min_in || !is_device_ptr(min_in) || !(cfl > 0.0)) return fail(SWE_ERR_ARG, "bad arguments");
    CU(cudaMemcpyAsync(&c->d_S->min_bits, min_in, sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
    launch(c, KIND_MISC, [&] { k_dt_finalize<<<1, 1, 0, c->stream>>>(c->d_S, cfl, 1); });
    c->min_valid = false;
    CU(cudaGetLastError());
    return SWE_OK;
}

static int check_stage(swe_ctx* c, int scheme, int stage) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (scheme < 0 || scheme > 3 || stage < 0 || stage > 1) return fail(SWE_ERR_ARG, "bad stage arguments");
    if (!c->has_zones) return fail(SWE_ERR_STATE, "no zones");
    if (scheme != K_HLLC && c->Z.nlayers < 2)
        return fail(SWE_ERR_STATE, "distributed MUSCL / WAF stages need zones with at least 2 ghost layers");
    const bool heun = scheme == K_MUSCL || scheme == K_MUSCL_MS;
    if (!heun && stage != 0) return fail(SWE_ERR_ARG, "Euler schemes have one stage");
    return SWE_OK;
}

int swe_dist_flux(swe_ctx* c, int scheme, int stage) {
    int rc = check_stage(c, scheme, stage); if (rc) return rc;
    Store& st = c->z;
    const double4* Uin = (stage == 0) ? st.A : st.B;
    run_grad(c, st, Uin, scheme);
    run_flux(c, st, Uin, scheme);
    CU(cudaGetLastError());
    return SWE_OK;
}

int swe_dist_update(swe_ctx* c, int scheme, int stage, int part) {
    int rc = check_stage(c, scheme, stage); if (rc) return rc;
    if (part < 0 || part > 2) return fail(SWE_ERR_ARG, "part must be 0 (all), 1 (send cells) or 2 (the rest)");
    const bool heun = scheme == K_MUSCL || scheme == K_MUSCL_MS;
    Store& st = c->z;
    if (heun && stage == 0) run_update(c, st, st.A, nullptr, st.B, 0, false, part);
    else if (heun) run_update(c, st, st.B, st.A, st.A, 1, true, part);
    else run_update(c, st, st.A, nullptr, st.A, 0, true, part);
    if ((!heun || stage == 1) && part != 1) { c->min_valid = true; c->steps++; }
    CU(cudaGetLastError());
    return SWE_OK;
}

int swe_dist_stage(swe_ctx* c, int scheme, int stage) {
    int rc = swe_dist_flux(c, scheme, stage); if (rc) return rc;
    return swe_dist_update(c, scheme, stage, 0);
}

int swe_get_time(swe_ctx* c, double* t_out, double* last_dt_out) {
    KeepMasks keep_masks(c);   // read-only
    if (check_ctx(c)) return SWE_ERR_ARG;
    StepScalars hs;
    CU(cudaMemcpyAsync(&hs, c->d_S, sizeof(hs), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    if (t_out) *t_out = hs.t;
    if (last_dt_out) *last_dt_out = hs.last_dt;
    return SWE_OK;
}

static int exchange_zone(swe_ctx* c, int zone, bool pack) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!c->has_zones) return fail(SWE_ERR_STATE, "no zones: call swe_zones_create first");
    if (zone < -1 || zone >= c->Z.nz) return fail(SWE_ERR_ARG, "zone out of range");
    if (zone == -1) {
        run_exchange_state(c, c->z.A, 0, c->nsend, pack, !pack);
    } else {
        for (size_t l = 0; l + 1 < c->Z.link_off.size(); ++l) {
            const int who = pack ? c->Z.link_src[l] : c->Z.link_dst[l];
            if (who != zone) continue;
            run_exchange_state(c, c->z.A, c->Z.link_off[l], c->Z.link_off[l + 1] - c->Z.link_off[l], pack, !pack);
        }
    }
    CU(cudaGetLastError());
    return SWE_OK;
}
int swe_pack_ghosts(swe_ctx* c, int zone) { return exchange_zone(c, zone, true); }
int swe_unpack_ghosts(swe_ctx* c, int zone) { return exchange_zone(c, zone, false); }

int swe_zone_stats(const swe_ctx* c, int64_t* send_cells_total, int64_t* bytes_per_exchange, int64_t* ghost_cells_total) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!c->has_zones) return fail(SWE_ERR_STATE, "no zones");
    int64_t gh = 0;
    for (const ZoneDesc& zd : c->Z.z) if (zd.offset >= 0) gh += zd.ncells - zd.nowned;
    if (send_cells_total) *send_cells_total = c->nsend;
    if (bytes_per_exchange) *bytes_per_exchange = c->nsend * 24;
    if (ghost_cells_total) *ghost_cells_total = gh;
    return SWE_OK;
}
int swe_zone_setup_ms(const swe_ctx* c, double* ghost_layers_ms, double* build_ms, double* total_ms) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!c->has_zones) return fail(SWE_ERR_STATE, "no zones");
    if (ghost_layers_ms) *ghost_layers_ms = c->zone_ms[0];
    if (build_ms) *build_ms = c->zone_ms[1];
    if (total_ms) *total_ms = c->zone_ms[2];
    return SWE_OK;
}
int swe_zone_setup_detail(const swe_ctx* c, double* ms /*5*/) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!c->has_zones) return fail(SWE_ERR_STATE, "no zones");
    if (!ms) return fail(SWE_ERR_ARG, "NULL output");
    ms[0] = c->zone_ms[3];                      // zone of every cell (RCB or the caller's array)
    ms[1] = c->zone_ms[0];                      // ghost layers of all zones on the device
    ms[2] = c->zone_ms[1] - c->zone_ms[3] - c->zone_ms[0];   // owned positions (device) + links and exchange lists (host)
    ms[3] = c->zone_ms[4] - c->zone_ms[1];      // the zones' arrays assembled on the device
    ms[4] = c->zone_ms[2];                      // whole call
    return SWE_OK;
}
int swe_zone_describe(const swe_ctx* c, int zone, int64_t* nowned, int64_t* nghost, int64_t* nlinks) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!c->has_zones || zone < 0 || zone >= c->Z.nz) return fail(SWE_ERR_ARG, "no such zone");
    const ZoneDesc& zd = c->Z.z[zone];
    if (nowned) *nowned = zd.nowned;
    if (nghost) *nghost = zd.ncells - zd.nowned;
    if (nlinks) *nlinks = (int64_t)zd.links.size();
    return SWE_OK;
}
// the zones' cell lists (source cell and layer of every cell of the concatenated mesh): one download,
// sliced per resident zone, the first time somebody asks
static int zone_cells_to_host(swe_ctx* c) {
    if (c->zone_cells_on_host) return SWE_OK;
    const size_t ncz = (size_t)c->z.nc;
    std::vector<int32_t> hsrc(ncz); std::vector<uint8_t> hlay(ncz);
    CU(cudaMemcpyAsync(hsrc.data(), c->d_src_of_cell, ncz * sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaMemcpyAsync(hlay.data(), c->z.dm.layer, ncz, cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    for (size_t r = 0; r < c->zr_zone.size(); ++r) {
        ZoneDesc& zd = c->Z.z[c->zr_zone[r]];
        zd.cells.assign(hsrc.begin() + c->zr_off[r], hsrc.begin() + c->zr_off[r] + zd.ncells);
        zd.layer.assign(hlay.begin() + c->zr_off[r], hlay.begin() + c->zr_off[r] + zd.ncells);
    }
    c->zone_cells_on_host = true;
    return SWE_OK;
}
int swe_zone_cells(const swe_ctx* cc, int zone, int32_t* cells, int32_t* layer) {
    swe_ctx* c = const_cast<swe_ctx*>(cc);
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!c->has_zones || zone < 0 || zone >= c->Z.nz) return fail(SWE_ERR_ARG, "no such zone");
    if (c->Z.zone_rank[zone] != c->Z.rank) return fail(SWE_ERR_ARG, "the zone lives on another rank");
    { int rc = zone_cells_to_host(c); if (rc) return rc; }
    const ZoneDesc& zd = c->Z.z[zone];
    for (size_t j = 0; j < zd.cells.size(); ++j) {
        if (cells) cells[j] = c->H.m.cell_user[zd.cells[j]];
        if (layer) layer[j] = zd.layer[j];
    }
    return SWE_OK;
}
int swe_zone_links(const swe_ctx* c, int zone, int32_t* src, int32_t* start, int32_t* count) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!c->has_zones || zone < 0 || zone >= c->Z.nz) return fail(SWE_ERR_ARG, "no such zone");
    const ZoneDesc& zd = c->Z.z[zone];
    for (size_t j = 0; j < zd.links.size(); ++j) {
        if (src) src[j] = zd.links[j].src;
        if (start) start[j] = zd.links[j].start;
        if (count) count[j] = zd.links[j].count;
    }
    return SWE_OK;
}
int swe_zone_sendlist(const swe_ctx* c, int zone, int link, int32_t* send_idx) {
    if (check_ctx(c)) return SWE_ERR_ARG;
    if (!c->has_zones || zone < 0 || zone >= c->Z.nz) return fail(SWE_ERR_ARG, "no such zone");
    const ZoneDesc& zd = c->Z.z[zone];
    if (link < 0 || link >= (int)zd.links.size() || !send_idx) return fail(SWE_ERR_ARG, "no such link");
    std::copy(zd.links[link].send.begin(), zd.links[link].send.end(), send_idx);
    return SWE_OK;
}

}  // extern "C"
