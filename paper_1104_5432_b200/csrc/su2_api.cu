// su2_api.cu — the C-ABI boundary (include/su2_heatbath.h): handle, argument
// checking, error capture, stream plumbing. No arithmetic of the method lives here.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include "../../include/su2_heatbath.h"
#include "su2_launch.h"

using namespace su2;

struct su2_lattice {
    Geom g;
    int precision;
    void* links;
    bool owns_links;
    cudaStream_t stream;
    uint64_t seed;
    bool initialised;
    Scratch sc;
    uint64_t launches;
    int last_substep;  // 2*mu+parity of the heat-bath sub-step that was the LAST work enqueued by this
                       // handle, else -1: decides whether the next sub-step may overlap it
    bool pdl;          // programmatic dependent launch enabled (su2_set_option SU2_OPT_OVERLAP)
    // su2_run: one step captured as a CUDA graph, replayed on a private stream
    cudaStream_t run_stream;
    cudaEvent_t run_ev_in, run_ev_out;
    cudaGraphExec_t run_exec;
    cudaGraphExec_t batch_exec;  // su2_batch_run: one round of the whole batch
    bool run_graphs;   // su2_run replays a captured CUDA graph (su2_set_option SU2_OPT_RUN_GRAPH)
    int tail_overlap;  // su2_run: the Polyakov kernel of a step runs beside the next step (SU2_OPT_TAIL_OVERLAP):
                       // 0 off, 1 on, -1 (default) automatic - see tail_overlap_on()
    cudaStream_t tail_stream;
    cudaEvent_t ev_fork, ev_join;
    int run_block;     // steps per captured graph (1, or kRunBlock with tail overlap)
    double creutz_below;  // [R15] su2_set_draw: 0 (KP), SU2_ALPHA_C (auto) or +inf (Creutz)
    // replica batch: nrep configurations one after the other from links_base; `links`,
    // `seed` and `initialised` are those of the selected replica (single-lattice calls act on it)
    int nrep, selected;
    void* links_base;
    size_t rep_bytes;
    uint64_t* rep_seed;        // [host] nrep
    unsigned char* rep_init;   // [host] nrep
    RepParams* rep_host;       // [host] nrep: what sc.reps holds
    // time slab of a lattice split over GPUs: local slices = 2 halo + Lt interior + 2 halo
    bool slab;
    int nt_glob, t0, Lt;     // global time extent, first global slice of the interior, interior slices
    SlabCtx sctx;            // peers (set by su2_slab_set_peers)
    bool peers_set;
    void* stage;       // canonical-order staging buffer of su2_get_links / su2_set_links (lazy, kept)
    int sticky;  // sticky error code
    char msg[256];
};

static int fail(su2_lattice* lat, int code, const char* what, cudaError_t ce = cudaSuccess)
{
    if (lat) {
        if (ce != cudaSuccess)
            snprintf(lat->msg, sizeof lat->msg, "%s: %s", what, cudaGetErrorString(ce));
        else
            snprintf(lat->msg, sizeof lat->msg, "%s", what);
        if (code == SU2_ECUDA) lat->sticky = code;
    }
    return code;
}
#define CK(lat, call)                                              \
    do {                                                           \
        cudaError_t ce__ = (call);                                 \
        if (ce__ != cudaSuccess) return fail(lat, SU2_ECUDA, #call, ce__); \
    } while (0)
#define ENTER(lat)                       \
    do {                                 \
        if (!(lat)) return SU2_EARG;     \
        if ((lat)->sticky) return (lat)->sticky; \
    } while (0)
// calls that step or measure a whole lattice by themselves: a slab needs its neighbours between sub-steps
#define NOT_ON_A_SLAB(lat, what)                                                                    \
    do {                                                                                            \
        if ((lat)->slab) return fail(lat, SU2_ESTATE, what ": not available on a slab handle (su2_slab_*)"); \
    } while (0)
// last_substep value after the Polyakov kernel of a step: sub-step (0,0) may overlap its tail
// (it waits for it like for a predecessor sub-step; that kernel itself waited for (3,1))
static const int kAfterStepTail = 8;
// every entry point that enqueues anything other than a heat-bath sub-step
#define NOT_A_SUBSTEP(lat) ((lat)->last_substep = -1)

// launch sub-step (mu, parity); it may overlap the tail of the previous launch only if
// that was its canonical predecessor [R4] on this handle
static void enqueue_substep(su2_lattice* lat, double beta, uint32_t sweep_idx, int mu, int parity,
                            double* epart = nullptr, const RunState* state = nullptr, cudaStream_t st = nullptr,
                            bool allow_overlap = true)
{
    const int idx = 2 * mu + parity;
    const bool overlap = allow_overlap && lat->pdl &&
                         (lat->last_substep == (idx + 7) % 8 || (idx == 0 && lat->last_substep == kAfterStepTail));
    if (!state) st = lat->stream;
    lat->launches += launch_heatbath_substep(lat->links, lat->g, lat->precision, mu, parity, beta,
                                             lat->creutz_below, lat->seed, sweep_idx, lat->sc.err, epart, state,
                                             overlap && !lat->slab, st, nullptr, 1, lat->slab ? &lat->sctx : nullptr);
    lat->last_substep = idx;
}

static bool valid_dims(int Nx, int Ny, int Nz, int Nt, int precision)
{
    const int n[4] = {Nx, Ny, Nz, Nt};
    uint64_t V = 1;
    for (int d = 0; d < 4; ++d) {
        if (n[d] < 2 || (n[d] & 1)) return false;
        V *= (uint64_t)n[d];
        if (V >= (1ull << 32)) return false;
    }
    return precision == 32 || precision == 64;
}

extern "C" size_t su2_lattice_bytes(int Nx, int Ny, int Nz, int Nt, int precision)
{
    if (!valid_dims(Nx, Ny, Nz, Nt, precision)) return 0;
    return (size_t)Nx * Ny * Nz * Nt * 4 * 4 * (precision == 32 ? sizeof(float) : sizeof(double));
}

// slab_Lt > 0: a time slab with slab_Lt interior slices (Nt = slab_Lt + 4 local slices)
static int create_impl(int Nx, int Ny, int Nz, int Nt, int precision, int nrep, void* dev_links, size_t bytes,
                       void* stream, bool external, su2_lattice** out, int slab_Lt = 0)
{
    if (!out) return SU2_EARG;
    *out = nullptr;
    if (!valid_dims(Nx, Ny, Nz, Nt, precision)) return SU2_EARG;
    // a batch indexes every link of every replica with 32 bits and puts the replica in grid y / z; a
    // single lattice indexes each of its 8 arrays separately (h < V/2), so V < 2^32 is its only limit
    if (nrep < 1 || nrep > 65535) return SU2_EARG;
    if (nrep > 1 && (uint64_t)nrep * 4ull * Nx * Ny * Nz * Nt >= (1ull << 32)) return SU2_EARG;
    const size_t rep_bytes = su2_lattice_bytes(Nx, Ny, Nz, Nt, precision);
    const size_t need = rep_bytes * (size_t)nrep;
    if (external && (!dev_links || bytes < need || ((uintptr_t)dev_links & 31))) return SU2_EARG;

    su2_lattice* lat = new (std::nothrow) su2_lattice;
    if (!lat) return SU2_EALLOC;
    memset(lat, 0, sizeof *lat);
    Geom& g = lat->g;
    g.n[0] = Nx; g.n[1] = Ny; g.n[2] = Nz; g.n[3] = Nt;
    g.nxh = Nx / 2;
    g.sy = g.nxh;
    g.sz = g.nxh * Ny;
    g.st = g.nxh * Ny * Nz;
    g.vh = (uint32_t)((uint64_t)Nx * Ny * Nz * Nt / 2);
    g.wup[0] = -(g.nxh - 1);
    g.wup[1] = -(Ny - 1) * g.sy;
    g.wup[2] = -(Nz - 1) * g.sz;
    g.wup[3] = -(Nt - 1) * g.st;
    g.t_lo = slab_Lt > 0 ? 2 : 0;
    g.nt_upd = slab_Lt > 0 ? slab_Lt : Nt;
    choose_tiling(g, nrep, precision);  // grid z holds (replica, z-t tile): falls back to the next shape / the linear launch
    lat->nrep = nrep;
    lat->rep_bytes = rep_bytes;
    lat->precision = precision;
    lat->last_substep = -1;
    lat->pdl = true;
    lat->run_graphs = true;
    lat->tail_overlap = -1;
    lat->stream = (cudaStream_t)stream;
    lat->owns_links = !external;
    lat->links = dev_links;
    lat->rep_seed = (uint64_t*)calloc((size_t)nrep, sizeof(uint64_t));
    lat->rep_init = (unsigned char*)calloc((size_t)nrep, 1);
    lat->rep_host = (RepParams*)calloc((size_t)nrep, sizeof(RepParams));
    if (!lat->rep_seed || !lat->rep_init || !lat->rep_host) {
        su2_lattice_destroy(lat);
        return SU2_EALLOC;
    }

    cudaError_t ce = cudaSuccess;
    if (!external) ce = cudaMalloc(&lat->links, need);
    const uint64_t v3 = (uint64_t)Nx * Ny * Nz;
    lat->sc.n_partials = partials_needed(g);
    if (ce == cudaSuccess) ce = cudaMalloc((void**)&lat->sc.partials, lat->sc.n_partials * sizeof(double));
    lat->links_base = lat->links;
    if (ce == cudaSuccess) ce = cudaMalloc((void**)&lat->sc.epart, 2 * (size_t)nrep * 3 * heatbath_ctas(g) * sizeof(double));
    if (ce == cudaSuccess) ce = cudaMalloc((void**)&lat->sc.field, (size_t)nrep * v3 * sizeof(double));
    if (ce == cudaSuccess) ce = cudaMalloc((void**)&lat->sc.reps, (size_t)nrep * sizeof(RepParams));
    if (ce == cudaSuccess) ce = cudaMalloc((void**)&lat->sc.out, (2 + kMaxR) * sizeof(double));
    if (ce == cudaSuccess) ce = cudaMalloc((void**)&lat->sc.state, 2 * kRunCopies * sizeof(RunState));
    if (ce == cudaSuccess) ce = cudaMalloc((void**)&lat->sc.slots, (size_t)nrep * 2 * (v3 / 64 + 1) * sizeof(double));
    if (ce == cudaSuccess) ce = cudaMalloc((void**)&lat->sc.ticket, ((size_t)nrep + 1) * sizeof(unsigned));
    if (ce == cudaSuccess) ce = cudaMemset(lat->sc.ticket, 0, ((size_t)nrep + 1) * sizeof(unsigned));
    if (ce == cudaSuccess) ce = cudaMalloc((void**)&lat->sc.err, sizeof(int));
    if (ce == cudaSuccess) ce = cudaMemset(lat->sc.err, 0, sizeof(int));
    if (ce != cudaSuccess) {
        const int code = (ce == cudaErrorMemoryAllocation) ? SU2_EALLOC : SU2_ECUDA;
        cudaGetLastError();
        su2_lattice_destroy(lat);
        return code;
    }
    *out = lat;
    return SU2_OK;
}

extern "C" int su2_lattice_create(int Nx, int Ny, int Nz, int Nt, int precision, su2_lattice** out)
{
    return create_impl(Nx, Ny, Nz, Nt, precision, 1, nullptr, 0, nullptr, false, out);
}

extern "C" int su2_lattice_create_batch(int Nx, int Ny, int Nz, int Nt, int precision, int n_replicas,
                                        su2_lattice** out)
{
    return create_impl(Nx, Ny, Nz, Nt, precision, n_replicas, nullptr, 0, nullptr, false, out);
}

extern "C" int su2_lattice_create_batch_external(int Nx, int Ny, int Nz, int Nt, int precision, int n_replicas,
                                                 void* dev_links, size_t bytes, void* cuda_stream, su2_lattice** out)
{
    return create_impl(Nx, Ny, Nz, Nt, precision, n_replicas, dev_links, bytes, cuda_stream, true, out);
}

extern "C" int su2_lattice_create_external(int Nx, int Ny, int Nz, int Nt, int precision, void* dev_links,
                                           size_t bytes, void* cuda_stream, su2_lattice** out)
{
    return create_impl(Nx, Ny, Nz, Nt, precision, 1, dev_links, bytes, cuda_stream, true, out);
}

extern "C" int su2_lattice_destroy(su2_lattice* lat)
{
    if (!lat) return SU2_OK;
    if (lat->owns_links && lat->links_base) cudaFree(lat->links_base);
    else if (lat->owns_links && lat->links) cudaFree(lat->links);
    if (lat->sc.reps) cudaFree(lat->sc.reps);
    free(lat->rep_seed);
    free(lat->rep_init);
    free(lat->rep_host);
    if (lat->sc.partials) cudaFree(lat->sc.partials);
    if (lat->sc.epart) cudaFree(lat->sc.epart);
    if (lat->sc.field) cudaFree(lat->sc.field);
    if (lat->sc.out) cudaFree(lat->sc.out);
    if (lat->stage) cudaFree(lat->stage);
    if (lat->sc.err) cudaFree(lat->sc.err);
    if (lat->sc.state) cudaFree(lat->sc.state);
    if (lat->sc.slots) cudaFree(lat->sc.slots);
    if (lat->sc.ticket) cudaFree(lat->sc.ticket);
    if (lat->run_exec) cudaGraphExecDestroy(lat->run_exec);
    if (lat->batch_exec) cudaGraphExecDestroy(lat->batch_exec);
    if (lat->run_ev_in) cudaEventDestroy(lat->run_ev_in);
    if (lat->run_ev_out) cudaEventDestroy(lat->run_ev_out);
    if (lat->run_stream) cudaStreamDestroy(lat->run_stream);
    if (lat->ev_fork) cudaEventDestroy(lat->ev_fork);
    if (lat->ev_join) cudaEventDestroy(lat->ev_join);
    if (lat->tail_stream) cudaStreamDestroy(lat->tail_stream);
    delete lat;
    return SU2_OK;
}

extern "C" int su2_set_stream(su2_lattice* lat, void* cuda_stream)
{
    ENTER(lat);
    NOT_A_SUBSTEP(lat);
    lat->stream = (cudaStream_t)cuda_stream;
    return SU2_OK;
}

// The captured step of su2_run holds what was current at capture: the link pointers of the selected
// replica, the expanded Philox keys of the seed, the draw's kernels. Whatever changes one of them drops it.
static void drop_run_graph(su2_lattice* lat)
{
    if (lat->run_exec) {
        cudaStreamSynchronize(lat->run_stream);
        cudaGraphExecDestroy(lat->run_exec);
        lat->run_exec = nullptr;
    }
    if (lat->batch_exec) {  // (seeds and couplings of a batch live in device memory: only the kernels are captured)
        cudaStreamSynchronize(lat->run_stream);
        cudaGraphExecDestroy(lat->batch_exec);
        lat->batch_exec = nullptr;
    }
}

extern "C" int su2_set_option(su2_lattice* lat, int option, int value)
{
    ENTER(lat);
    NOT_A_SUBSTEP(lat);
    if (value != 0 && value != 1) return fail(lat, SU2_EARG, "su2_set_option: value must be 0 or 1");
    switch (option) {
        case SU2_OPT_OVERLAP: lat->pdl = value != 0; break;
        case SU2_OPT_RUN_GRAPH: lat->run_graphs = value != 0; break;
        case SU2_OPT_TAIL_OVERLAP: lat->tail_overlap = value != 0 ? 1 : 0; break;
        default: return fail(lat, SU2_EARG, "su2_set_option: unknown option");
    }
    drop_run_graph(lat);  // the captured step was built with the other setting
    return SU2_OK;
}

extern "C" int su2_init(su2_lattice* lat, int start, uint64_t seed)
{
    ENTER(lat);
    NOT_A_SUBSTEP(lat);
    if (start != SU2_START_COLD && start != SU2_START_HOT) return fail(lat, SU2_EARG, "su2_init: bad start");
    // a slab draws every local slice, halos included, from the global site it is a copy of
    lat->launches += launch_init(lat->links, lat->g, lat->precision, start, seed, lat->stream,
                                 lat->slab ? lat->t0 - 2 : 0, lat->slab ? lat->nt_glob : 0);
    CK(lat, cudaGetLastError());
    if (seed != lat->seed) drop_run_graph(lat);  // its kernels carry the old seed's round keys
    lat->seed = seed;
    lat->initialised = true;
    lat->rep_seed[lat->selected] = seed;
    lat->rep_init[lat->selected] = 1;
    return SU2_OK;
}

extern "C" int su2_set_seed(su2_lattice* lat, uint64_t seed)
{
    ENTER(lat);
    if (seed != lat->seed) drop_run_graph(lat);  // its kernels carry the old seed's round keys
    lat->seed = seed;
    lat->rep_seed[lat->selected] = seed;
    return SU2_OK;
}

extern "C" int su2_replicas(const su2_lattice* lat) { return lat ? lat->nrep : 0; }

extern "C" int su2_select_replica(su2_lattice* lat, int replica)
{
    ENTER(lat);
    NOT_A_SUBSTEP(lat);
    if (replica < 0 || replica >= lat->nrep) return fail(lat, SU2_EARG, "su2_select_replica: no such replica");
    if (replica != lat->selected) drop_run_graph(lat);
    lat->selected = replica;
    lat->links = (char*)lat->links_base + (size_t)replica * lat->rep_bytes;
    lat->seed = lat->rep_seed[replica];
    lat->initialised = lat->rep_init[replica] != 0;
    return SU2_OK;
}

extern "C" int su2_batch_init(su2_lattice* lat, int start, const uint64_t* seeds)
{
    ENTER(lat);
    NOT_A_SUBSTEP(lat);
    if (start != SU2_START_COLD && start != SU2_START_HOT) return fail(lat, SU2_EARG, "su2_batch_init: bad start");
    if (!seeds) return fail(lat, SU2_EARG, "su2_batch_init: NULL seeds");
    drop_run_graph(lat);
    for (int r = 0; r < lat->nrep; ++r) {
        lat->launches += launch_init((char*)lat->links_base + (size_t)r * lat->rep_bytes, lat->g, lat->precision, start,
                                     seeds[r], lat->stream);
        lat->rep_seed[r] = seeds[r];
        lat->rep_init[r] = 1;
    }
    CK(lat, cudaGetLastError());
    lat->seed = lat->rep_seed[lat->selected];
    lat->initialised = true;
    return SU2_OK;
}

// One step of every replica in 9 launches: the 8 sub-steps over the whole batch (ALT
// kernels, replica = leading part of the grid, 1/beta and seed per replica from device memory), then
// the Polyakov kernel with one step tail per replica.
extern "C" int su2_batch_sweep_measure(su2_lattice* lat, const double* betas, uint32_t sweep_idx, double* dev_out,
                                       size_t index)
{
    ENTER(lat);
    NOT_ON_A_SLAB(lat, "su2_batch_sweep_measure");
    NOT_A_SUBSTEP(lat);
    if (!betas || !dev_out) return fail(lat, SU2_EARG, "su2_batch_sweep_measure: NULL argument");
    bool changed = false;
    for (int r = 0; r < lat->nrep; ++r) {
        if (!(betas[r] > 0.0) || !isfinite(betas[r])) return fail(lat, SU2_EARG, "beta must be finite and > 0");
        if (!lat->rep_init[r]) return fail(lat, SU2_ESTATE, "a replica of the batch is not initialised");
        const RepParams rp = {1.0 / betas[r], lat->rep_seed[r]};
        changed = changed || rp.inv_beta != lat->rep_host[r].inv_beta || rp.seed != lat->rep_host[r].seed;
        lat->rep_host[r] = rp;
    }
    if (changed) {  // rare: the kernels of earlier steps must have read the old values first
        CK(lat, cudaStreamSynchronize(lat->stream));
        CK(lat, cudaMemcpyAsync(lat->sc.reps, lat->rep_host, (size_t)lat->nrep * sizeof(RepParams),
                                cudaMemcpyHostToDevice, lat->stream));
    }
    const size_t ctas = heatbath_ctas(lat->g);
    int prev = -1;
    for (int mu = 0; mu < 4; ++mu)
        for (int p = 0; p < 2; ++p) {
            const int idx = 2 * mu + p;
            const bool overlap = lat->pdl && prev == (idx + 7) % 8;
            lat->launches += launch_heatbath_substep(
                lat->links_base, lat->g, lat->precision, mu, p, 1.0, lat->creutz_below, 0, sweep_idx, lat->sc.err,
                (p == 1 && mu >= 1) ? lat->sc.epart + (mu - 1) * ctas : nullptr, nullptr, overlap, lat->stream,
                lat->sc.reps, lat->nrep);
            prev = idx;
        }
    lat->launches += launch_polyakov_step(lat->links_base, lat->g, lat->precision, lat->sc, lat->sc.epart, 3 * ctas,
                                          1.0 / (6.0 * 2.0 * (double)lat->g.vh),
                                          dev_out + 2 * index * (size_t)lat->nrep, nullptr, lat->pdl, lat->stream,
                                          lat->nrep);
    CK(lat, cudaGetLastError());
    return SU2_OK;
}

// one round of the whole batch on stream `st`, sweep index and output slot read from the device RunState
static void enqueue_batch_round(su2_lattice* lat, cudaStream_t st, bool allow_overlap)
{
    const size_t ctas = heatbath_ctas(lat->g);
    int prev = -1;
    for (int mu = 0; mu < 4; ++mu)
        for (int p = 0; p < 2; ++p) {
            const int idx = 2 * mu + p;
            const bool overlap = allow_overlap && lat->pdl && prev == (idx + 7) % 8;
            lat->launches += launch_heatbath_substep(
                lat->links_base, lat->g, lat->precision, mu, p, 1.0, lat->creutz_below, 0, 0u, lat->sc.err,
                (p == 1 && mu >= 1) ? lat->sc.epart + (mu - 1) * ctas : nullptr, lat->sc.state, overlap, st, lat->sc.reps,
                lat->nrep);
            prev = idx;
        }
    lat->launches += launch_polyakov_step(lat->links_base, lat->g, lat->precision, lat->sc, lat->sc.epart, 3 * ctas,
                                          1.0 / (6.0 * 2.0 * (double)lat->g.vh), nullptr, lat->sc.state,
                                          allow_overlap && lat->pdl, st, lat->nrep);
}

// su2_run's counterpart for a batch: n rounds of su2_batch_sweep_measure as one call; one round is
// captured as a CUDA graph and replayed, sweep index and output slot live in the device loop state.
extern "C" int su2_batch_run(su2_lattice* lat, const double* betas, uint32_t sweep_idx0, uint32_t n_steps, double* dev_out)
{
    ENTER(lat);
    NOT_ON_A_SLAB(lat, "su2_batch_run");
    NOT_A_SUBSTEP(lat);
    if (!betas || (!dev_out && n_steps)) return fail(lat, SU2_EARG, "su2_batch_run: NULL argument");
    bool changed = false;
    for (int r = 0; r < lat->nrep; ++r) {
        if (!(betas[r] > 0.0) || !isfinite(betas[r])) return fail(lat, SU2_EARG, "beta must be finite and > 0");
        if (!lat->rep_init[r]) return fail(lat, SU2_ESTATE, "a replica of the batch is not initialised");
        const RepParams rp = {1.0 / betas[r], lat->rep_seed[r]};
        changed = changed || rp.inv_beta != lat->rep_host[r].inv_beta || rp.seed != lat->rep_host[r].seed;
        lat->rep_host[r] = rp;
    }
    if (n_steps == 0) return SU2_OK;
    if (changed) {  // rare: the kernels of earlier steps must have read the old values first
        CK(lat, cudaStreamSynchronize(lat->stream));
        CK(lat, cudaMemcpyAsync(lat->sc.reps, lat->rep_host, (size_t)lat->nrep * sizeof(RepParams),
                                cudaMemcpyHostToDevice, lat->stream));
    }
    if (!lat->run_stream) {
        CK(lat, cudaStreamCreateWithFlags(&lat->run_stream, cudaStreamNonBlocking));
        CK(lat, cudaEventCreateWithFlags(&lat->run_ev_in, cudaEventDisableTiming));
        CK(lat, cudaEventCreateWithFlags(&lat->run_ev_out, cudaEventDisableTiming));
    }
    CK(lat, cudaEventRecord(lat->run_ev_in, lat->stream));
    CK(lat, cudaStreamWaitEvent(lat->run_stream, lat->run_ev_in, 0));
    lat->launches += launch_set_run_state(lat->sc.state, 1.0, dev_out, sweep_idx0, 0u, lat->run_stream);
    if (lat->run_graphs && !lat->batch_exec) {
        for (int attempt = 0; attempt < 2 && !lat->batch_exec; ++attempt) {
            const uint64_t launches0 = lat->launches;
            cudaGraph_t graph = nullptr;
            if (cudaStreamBeginCapture(lat->run_stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) break;
            enqueue_batch_round(lat, lat->run_stream, attempt == 0);
            cudaError_t ce = cudaStreamEndCapture(lat->run_stream, &graph);
            lat->launches = launches0;  // captured, not launched
            if (ce == cudaSuccess && graph) ce = cudaGraphInstantiate(&lat->batch_exec, graph, 0);
            if (graph) cudaGraphDestroy(graph);
            if (ce != cudaSuccess) {
                lat->batch_exec = nullptr;
                cudaGetLastError();
            }
        }
    }
    for (uint32_t i = 0; i < n_steps; ++i) {
        if (lat->run_graphs && lat->batch_exec) {
            CK(lat, cudaGraphLaunch(lat->batch_exec, lat->run_stream));
            lat->launches += 9;
        } else {
            enqueue_batch_round(lat, lat->run_stream, true);
        }
    }
    CK(lat, cudaGetLastError());
    CK(lat, cudaEventRecord(lat->run_ev_out, lat->run_stream));
    CK(lat, cudaStreamWaitEvent(lat->stream, lat->run_ev_out, 0));
    return SU2_OK;
}

extern "C" int su2_set_draw(su2_lattice* lat, int method)
{
    ENTER(lat);
    NOT_A_SUBSTEP(lat);
    double cb;
    switch (method) {
        case SU2_DRAW_KP: cb = 0.0; break;
        case SU2_DRAW_AUTO: cb = SU2_ALPHA_C; break;
        case SU2_DRAW_CREUTZ: cb = INFINITY; break;
        default: return fail(lat, SU2_EARG, "su2_set_draw: bad method");
    }
    if (cb != lat->creutz_below) drop_run_graph(lat);  // the captured step holds the other kernels
    lat->creutz_below = cb;
    return SU2_OK;
}

static int check_beta(su2_lattice* lat, double beta)
{
    if (!(beta > 0.0) || !isfinite(beta)) return fail(lat, SU2_EARG, "beta must be finite and > 0");
    if (!lat->initialised) return fail(lat, SU2_ESTATE, "lattice not initialised (su2_init / su2_set_links)");
    return SU2_OK;
}

extern "C" int su2_heatbath_substep(su2_lattice* lat, double beta, uint32_t sweep_idx, int mu, int parity)
{
    ENTER(lat);
    if (int rc = check_beta(lat, beta)) return rc;
    if (mu < 0 || mu > 3 || (parity != 0 && parity != 1)) return fail(lat, SU2_EARG, "bad mu / parity");
    if (lat->slab && !lat->peers_set) return fail(lat, SU2_ESTATE, "slab: su2_slab_set_peers first");
    enqueue_substep(lat, beta, sweep_idx, mu, parity);
    CK(lat, cudaGetLastError());
    return SU2_OK;
}

extern "C" int su2_heatbath_sweep(su2_lattice* lat, double beta, uint32_t sweep_idx)
{
    ENTER(lat);
    NOT_ON_A_SLAB(lat, "su2_heatbath_sweep");
    if (int rc = check_beta(lat, beta)) return rc;
    for (int mu = 0; mu < 4; ++mu)      // [R4] direction outer,
        for (int p = 0; p < 2; ++p)     //      parity inner
            enqueue_substep(lat, beta, sweep_idx, mu, p);
    CK(lat, cudaGetLastError());
    return SU2_OK;
}

extern "C" int su2_heatbath_sweep_measure(su2_lattice* lat, double beta, uint32_t sweep_idx, double* dev_out,
                                          size_t index, void* event_after_sweep)
{
    ENTER(lat);
    NOT_ON_A_SLAB(lat, "su2_heatbath_sweep_measure");
    if (int rc = check_beta(lat, beta)) return rc;
    if (!dev_out) return fail(lat, SU2_EARG, "su2_heatbath_sweep_measure: NULL dev_out");
    const size_t ctas = heatbath_ctas(lat->g);
    for (int mu = 0; mu < 4; ++mu)
        for (int p = 0; p < 2; ++p)
            enqueue_substep(lat, beta, sweep_idx, mu, p, (p == 1 && mu >= 1) ? lat->sc.epart + (mu - 1) * ctas : nullptr);
    if (event_after_sweep) CK(lat, cudaEventRecord((cudaEvent_t)event_after_sweep, lat->stream));
    // the three partial sets cover every plaquette of the new configuration once;
    // the Polyakov kernel also finishes both sums and, like a sub-step, may be
    // scheduled while its predecessor (3,1) drains; the next sweep's (0,0) may follow it the same way
    lat->launches += launch_polyakov_step(lat->links, lat->g, lat->precision, lat->sc, lat->sc.epart, 3 * ctas,
                                          1.0 / (6.0 * 2.0 * (double)lat->g.vh), dev_out + 2 * index, nullptr,
                                          lat->pdl && !event_after_sweep, lat->stream);
    lat->last_substep = kAfterStepTail;
    CK(lat, cudaGetLastError());
    return SU2_OK;
}

// Automatic choice: on wherever a sub-step is a few CTA waves - every lattice that does not take
// the walk (g.tloop == 1: below ~5 M sites) - where it is worth 5-23 % of a step and never costs; off on the large
// lattices, where forcing sub-step (3,0) behind two predecessors costs 4 %.
static bool tail_overlap_on(const su2_lattice* lat)
{
    return lat->tail_overlap < 0 ? lat->g.tloop == 1 : lat->tail_overlap != 0;
}

// Steps of su2_run on stream `st`, every per-step quantity read from a device RunState.
// Plain mode (tail_st == NULL): 8 sub-steps + the Polyakov kernel with the step tail, all on `st`, one loop state.
// Tail overlap: the Polyakov kernel reads only U_t, which the next step does not write before its
// sub-step (3,0), so it runs on `tail_st` beside the next step's first six sub-steps: forked behind (3,1), joined
// before the next (3,0). What the two then touch at the same time alternates between two sets by step parity:
// the fused-plaquette partials (written by (1,1), (2,1), (3,1), read by the tail) and the loop state (read by the
// sub-steps, advanced - by 2 - by the tail). Same kernels on the same inputs: bit-identical results.
#ifndef SU2_RUN_BLOCK
#define SU2_RUN_BLOCK 16
#endif
static const int kRunBlock = SU2_RUN_BLOCK;  // steps per captured graph with tail overlap (graph launches serialise: the last
                                              // tail of a block is not overlapped; 4 / 8 / 16 / 32 measured, profiles/r02b.md)
static void enqueue_run_steps(su2_lattice* lat, cudaStream_t st, cudaStream_t tail_st, int count, bool allow_overlap)
{
    const size_t ctas = heatbath_ctas(lat->g);
    const double scale = 1.0 / (6.0 * 2.0 * (double)lat->g.vh);
    bool pending_join = false;
    for (int i = 0; i < count; ++i) {
        const int e = tail_st ? (i & 1) : 0;
        double* epart = lat->sc.epart + (size_t)e * 3 * ctas;
        RunState* state = lat->sc.state + (size_t)e * kRunCopies;
        lat->last_substep = -1;
        for (int mu = 0; mu < 4; ++mu)
            for (int p = 0; p < 2; ++p) {
                bool ov = allow_overlap;
                if (tail_st && mu == 3 && p == 0 && pending_join) {  // the previous tail still reads U_t
                    cudaStreamWaitEvent(st, lat->ev_join, 0);
                    pending_join = false;
                    ov = false;  // two predecessors: launched fully serialised
                }
                enqueue_substep(lat, 1.0, 0u, mu, p, (p == 1 && mu >= 1) ? epart + (mu - 1) * ctas : nullptr, state, st, ov);
            }
        if (tail_st) {
            cudaEventRecord(lat->ev_fork, st);
            cudaStreamWaitEvent(tail_st, lat->ev_fork, 0);
            lat->launches += launch_polyakov_step(lat->links, lat->g, lat->precision, lat->sc, epart, 3 * ctas, scale,
                                                  nullptr, state, false, tail_st, 1, 2u);
            cudaEventRecord(lat->ev_join, tail_st);
            pending_join = true;
            lat->last_substep = 7;  // the next (0,0) follows (3,1) on `st`
        } else {
            lat->launches += launch_polyakov_step(lat->links, lat->g, lat->precision, lat->sc, epart, 3 * ctas, scale,
                                                  nullptr, state, allow_overlap && lat->pdl, st);
            lat->last_substep = kAfterStepTail;
        }
    }
    if (pending_join) cudaStreamWaitEvent(st, lat->ev_join, 0);
    lat->last_substep = -1;
}

// capture `count` steps into an executable graph; with programmatic edges first, without if the
// driver refuses them
static bool build_run_graph(su2_lattice* lat, int count)
{
    cudaStream_t tail = tail_overlap_on(lat) ? lat->tail_stream : nullptr;
    for (int attempt = 0; attempt < 2 && !lat->run_exec; ++attempt) {
        const bool overlap = attempt == 0;
        const uint64_t launches0 = lat->launches;
        cudaGraph_t graph = nullptr;
        if (cudaStreamBeginCapture(lat->run_stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) break;
        enqueue_run_steps(lat, lat->run_stream, tail, count, overlap);
        cudaError_t ce = cudaStreamEndCapture(lat->run_stream, &graph);
        lat->launches = launches0;  // captured, not launched
        if (ce == cudaSuccess && graph) ce = cudaGraphInstantiate(&lat->run_exec, graph, 0);
        if (graph) cudaGraphDestroy(graph);
        if (ce != cudaSuccess) {
            lat->run_exec = nullptr;
            cudaGetLastError();
        }
    }
    lat->run_block = count;
    return lat->run_exec != nullptr;
}

extern "C" int su2_run(su2_lattice* lat, double beta, uint32_t sweep_idx0, uint32_t n_steps, double* dev_out)
{
    ENTER(lat);
    NOT_ON_A_SLAB(lat, "su2_run");
    NOT_A_SUBSTEP(lat);
    if (int rc = check_beta(lat, beta)) return rc;
    if (!dev_out && n_steps) return fail(lat, SU2_EARG, "su2_run: NULL dev_out");
    if (n_steps == 0) return SU2_OK;
    if (!lat->run_stream) {
        CK(lat, cudaStreamCreateWithFlags(&lat->run_stream, cudaStreamNonBlocking));
        CK(lat, cudaEventCreateWithFlags(&lat->run_ev_in, cudaEventDisableTiming));
        CK(lat, cudaEventCreateWithFlags(&lat->run_ev_out, cudaEventDisableTiming));
    }
    if (tail_overlap_on(lat) && !lat->tail_stream) {
        CK(lat, cudaStreamCreateWithFlags(&lat->tail_stream, cudaStreamNonBlocking));
        CK(lat, cudaEventCreateWithFlags(&lat->ev_fork, cudaEventDisableTiming));
        CK(lat, cudaEventCreateWithFlags(&lat->ev_join, cudaEventDisableTiming));
    }
    cudaStream_t tail = tail_overlap_on(lat) ? lat->tail_stream : nullptr;
    // the private stream continues the handle's stream and hands back to it
    CK(lat, cudaEventRecord(lat->run_ev_in, lat->stream));
    CK(lat, cudaStreamWaitEvent(lat->run_stream, lat->run_ev_in, 0));
    // loop state: one set, or two alternating by step parity (set e starts at step e and advances by 2)
    lat->launches += launch_set_run_state(lat->sc.state, 1.0 / beta, dev_out, sweep_idx0, 0u, lat->run_stream);
    if (tail)
        lat->launches += launch_set_run_state(lat->sc.state + kRunCopies, 1.0 / beta, dev_out, sweep_idx0 + 1u, 1u,
                                              lat->run_stream);
    const int block = tail ? kRunBlock : 1;
    const bool graphs = lat->run_graphs && (lat->run_exec || build_run_graph(lat, block));
    const uint64_t per_step = 8 + 1;
    uint32_t done = 0;
    if (graphs)
        for (; done + (uint32_t)block <= n_steps; done += (uint32_t)block) {
            CK(lat, cudaGraphLaunch(lat->run_exec, lat->run_stream));
            lat->launches += per_step * (uint64_t)block;
        }
    // the remainder of a block (or everything, without graphs) is enqueued directly; a block is an even number of
    // steps, so the parity of the remaining steps starts at 0 again
    if (done < n_steps) enqueue_run_steps(lat, lat->run_stream, tail, (int)(n_steps - done), true);
    CK(lat, cudaGetLastError());
    CK(lat, cudaEventRecord(lat->run_ev_out, lat->run_stream));
    CK(lat, cudaStreamWaitEvent(lat->stream, lat->run_ev_out, 0));
    return SU2_OK;
}

// synchronise and surface device-side flags
static int sync_and_check(su2_lattice* lat)
{
    int flags = 0;
    CK(lat, cudaMemcpyAsync(&flags, lat->sc.err, sizeof(int), cudaMemcpyDeviceToHost, lat->stream));
    CK(lat, cudaStreamSynchronize(lat->stream));
    if (flags & 1) return fail(lat, SU2_ECUDA, "Kennedy-Pendleton trial cap (10000) hit: alpha = beta*k too small");
    if (flags & 2) return fail(lat, SU2_ECUDA, "bounds check (HB_BOUNDS_CHECK build): a link index left its array");
    return SU2_OK;
}

extern "C" int su2_synchronize(su2_lattice* lat)
{
    ENTER(lat);
    NOT_A_SUBSTEP(lat);
    return sync_and_check(lat);
}

extern "C" int su2_measure_async(su2_lattice* lat, double* dev_out, size_t index)
{
    ENTER(lat);
    NOT_ON_A_SLAB(lat, "su2_measure_async");
    NOT_A_SUBSTEP(lat);
    if (!dev_out) return fail(lat, SU2_EARG, "su2_measure_async: NULL dev_out");
    if (!lat->initialised) return fail(lat, SU2_ESTATE, "lattice not initialised");
    lat->launches += launch_plaquette(lat->links, lat->g, lat->precision, lat->sc, dev_out + 2 * index, lat->stream);
    lat->launches +=
        launch_polyakov(lat->links, lat->g, lat->precision, lat->sc, dev_out + 2 * index + 1, lat->stream);
    CK(lat, cudaGetLastError());
    return SU2_OK;
}

extern "C" int su2_measure(su2_lattice* lat, double* plaquette_out, double* polyakov_out)
{
    ENTER(lat);
    NOT_ON_A_SLAB(lat, "su2_measure");
    NOT_A_SUBSTEP(lat);
    if (!lat->initialised) return fail(lat, SU2_ESTATE, "lattice not initialised");
    if (plaquette_out)
        lat->launches += launch_plaquette(lat->links, lat->g, lat->precision, lat->sc, lat->sc.out, lat->stream);
    if (polyakov_out)
        lat->launches += launch_polyakov(lat->links, lat->g, lat->precision, lat->sc, lat->sc.out + 1, lat->stream);
    CK(lat, cudaGetLastError());
    double host[2] = {0, 0};
    CK(lat, cudaMemcpyAsync(host, lat->sc.out, sizeof host, cudaMemcpyDeviceToHost, lat->stream));
    if (int rc = sync_and_check(lat)) return rc;
    if (plaquette_out) *plaquette_out = host[0];
    if (polyakov_out) *polyakov_out = host[1];
    return SU2_OK;
}

extern "C" int su2_mean_plaquette(su2_lattice* lat, double* out)
{
    if (!out) return lat ? fail(lat, SU2_EARG, "NULL out") : SU2_EARG;
    return su2_measure(lat, out, nullptr);
}

extern "C" int su2_polyakov_loop(su2_lattice* lat, double* out)
{
    if (!out) return lat ? fail(lat, SU2_EARG, "NULL out") : SU2_EARG;
    return su2_measure(lat, nullptr, out);
}

extern "C" int su2_polyakov_correlator(su2_lattice* lat, int rmax, double* out)
{
    ENTER(lat);
    NOT_ON_A_SLAB(lat, "su2_polyakov_correlator");
    NOT_A_SUBSTEP(lat);
    if (!out) return fail(lat, SU2_EARG, "NULL out");
    if (!lat->initialised) return fail(lat, SU2_ESTATE, "lattice not initialised");
    int nmin = lat->g.n[0] < lat->g.n[1] ? lat->g.n[0] : lat->g.n[1];
    if (lat->g.n[2] < nmin) nmin = lat->g.n[2];
    if (rmax < 1 || rmax > nmin / 2 || rmax > kMaxR) return fail(lat, SU2_EARG, "rmax out of range");
    lat->launches += launch_polyakov(lat->links, lat->g, lat->precision, lat->sc, lat->sc.out + 1, lat->stream);
    lat->launches += launch_polyakov_correlator(lat->g, lat->sc, rmax, lat->sc.out + 2, lat->stream);
    CK(lat, cudaGetLastError());
    CK(lat, cudaMemcpyAsync(out, lat->sc.out + 2, rmax * sizeof(double), cudaMemcpyDeviceToHost, lat->stream));
    return sync_and_check(lat);
}

extern "C" int su2_get_links(su2_lattice* lat, void* host_dst, size_t bytes)
{
    ENTER(lat);
    NOT_A_SUBSTEP(lat);
    const Geom& g = lat->g;
    const size_t need = su2_lattice_bytes(g.n[0], g.n[1], g.n[2], g.n[3], lat->precision);
    if (!host_dst || bytes != need) return fail(lat, SU2_EARG, "su2_get_links: bad buffer");
    if (!lat->initialised) return fail(lat, SU2_ESTATE, "lattice not initialised");
    if (!lat->stage && cudaMalloc(&lat->stage, need) != cudaSuccess) {
        cudaGetLastError();
        lat->stage = nullptr;
        return fail(lat, SU2_EALLOC, "su2_get_links: staging buffer");
    }
    void* stage = lat->stage;
    lat->launches += launch_to_canonical(lat->links, stage, g, lat->precision, lat->stream);
    cudaError_t ce = cudaGetLastError();
    if (ce == cudaSuccess) ce = cudaMemcpyAsync(host_dst, stage, need, cudaMemcpyDeviceToHost, lat->stream);
    if (ce != cudaSuccess) return fail(lat, SU2_ECUDA, "su2_get_links", ce);
    return sync_and_check(lat);  // the links of a run that raised a device-side flag are not handed out silently
}

extern "C" int su2_set_links(su2_lattice* lat, const void* host_src, size_t bytes)
{
    ENTER(lat);
    NOT_A_SUBSTEP(lat);
    const Geom& g = lat->g;
    const size_t need = su2_lattice_bytes(g.n[0], g.n[1], g.n[2], g.n[3], lat->precision);
    if (!host_src || bytes != need) return fail(lat, SU2_EARG, "su2_set_links: bad buffer");
    if (!lat->stage && cudaMalloc(&lat->stage, need) != cudaSuccess) {
        cudaGetLastError();
        lat->stage = nullptr;
        return fail(lat, SU2_EALLOC, "su2_set_links: staging buffer");
    }
    void* stage = lat->stage;
    cudaError_t ce = cudaMemcpyAsync(stage, host_src, need, cudaMemcpyHostToDevice, lat->stream);
    if (ce == cudaSuccess) {
        lat->launches += launch_to_device_layout(stage, lat->links, g, lat->precision, lat->stream);
        ce = cudaGetLastError();
    }
    if (ce == cudaSuccess) ce = cudaStreamSynchronize(lat->stream);
    if (ce != cudaSuccess) return fail(lat, SU2_ECUDA, "su2_set_links", ce);
    lat->initialised = true;
    lat->rep_init[lat->selected] = 1;
    return SU2_OK;
}

// ---------------------------------------------------------------------------- time slabs
static bool valid_slab(int Nx, int Ny, int Nz, int Nt, int precision, int t0, int Lt)
{
    if (!valid_dims(Nx, Ny, Nz, Nt, precision)) return false;
    if (Lt < 2 || (Lt & 1) || t0 < 0 || (t0 & 1) || t0 + Lt > Nt) return false;
    return valid_dims(Nx, Ny, Nz, Lt + 4, precision);
}

extern "C" size_t su2_slab_bytes(int Nx, int Ny, int Nz, int Lt, int precision)
{
    if (Lt < 2 || (Lt & 1)) return 0;
    return su2_lattice_bytes(Nx, Ny, Nz, Lt + 4, precision);
}

static int slab_create(int Nx, int Ny, int Nz, int Nt, int precision, int t0, int Lt, void* dev_links, size_t bytes,
                       void* stream, bool external, su2_lattice** out)
{
    if (!out) return SU2_EARG;
    *out = nullptr;
    if (!valid_slab(Nx, Ny, Nz, Nt, precision, t0, Lt)) return SU2_EARG;
    const int rc = create_impl(Nx, Ny, Nz, Lt + 4, precision, 1, dev_links, bytes, stream, external, out, Lt);
    if (rc != SU2_OK) return rc;
    su2_lattice* lat = *out;
    lat->slab = true;
    lat->nt_glob = Nt;
    lat->t0 = t0;
    lat->Lt = Lt;
    // local slice t holds global slice t0 - 2 + t: site indices differ by (t0 - 2) * NxNyNz (mod 2^32)
    lat->sctx.s_off = (uint32_t)((int64_t)(t0 - 2) * (int64_t)(2 * lat->g.st));
    return SU2_OK;
}

extern "C" int su2_slab_create(int Nx, int Ny, int Nz, int Nt, int precision, int t0, int Lt, su2_lattice** out)
{
    return slab_create(Nx, Ny, Nz, Nt, precision, t0, Lt, nullptr, 0, nullptr, false, out);
}

extern "C" int su2_slab_create_external(int Nx, int Ny, int Nz, int Nt, int precision, int t0, int Lt, void* dev_links,
                                        size_t bytes, void* cuda_stream, su2_lattice** out)
{
    return slab_create(Nx, Ny, Nz, Nt, precision, t0, Lt, dev_links, bytes, cuda_stream, true, out);
}

extern "C" int su2_slab_set_peers(su2_lattice* lat, void* lo_links, int lo_Lt, void* hi_links, int hi_Lt)
{
    ENTER(lat);
    NOT_A_SUBSTEP(lat);
    if (!lat->slab) return fail(lat, SU2_ESTATE, "su2_slab_set_peers: not a slab handle");
    if (!lo_links || !hi_links || lo_Lt < 2 || (lo_Lt & 1) || hi_Lt < 2 || (hi_Lt & 1))
        return fail(lat, SU2_EARG, "su2_slab_set_peers: bad argument");
    SlabCtx& c = lat->sctx;
    c.peer_lo = lo_links;
    c.peer_hi = hi_links;
    c.vh_lo = (uint32_t)(lat->g.st * (lo_Lt + 4));
    c.vh_hi = (uint32_t)(lat->g.st * (hi_Lt + 4));
    c.d_lo = lo_Lt * lat->g.st;    // own slice 2      -> slice lo_Lt + 2 (upper halo) of the slab below
    c.d_hi = -lat->Lt * lat->g.st; // own slice Lt + 1 -> slice 1 (lower halo) of the slab above
    lat->peers_set = true;
    return SU2_OK;
}

extern "C" int su2_slab_substep(su2_lattice* lat, double beta, uint32_t sweep_idx, int mu, int parity, int fuse_plaquette)
{
    ENTER(lat);
    if (!lat->slab) return fail(lat, SU2_ESTATE, "su2_slab_substep: not a slab handle");
    if (int rc = check_beta(lat, beta)) return rc;
    if (mu < 0 || mu > 3 || (parity != 0 && parity != 1)) return fail(lat, SU2_EARG, "bad mu / parity");
    if (!lat->peers_set) return fail(lat, SU2_ESTATE, "slab: su2_slab_set_peers first");
    const size_t ctas = heatbath_ctas(lat->g);
    enqueue_substep(lat, beta, sweep_idx, mu, parity,
                    (fuse_plaquette && parity == 1 && mu >= 1) ? lat->sc.epart + (mu - 1) * ctas : nullptr);
    CK(lat, cudaGetLastError());
    return SU2_OK;
}

extern "C" int su2_slab_plaquette(su2_lattice* lat, int fused, double* dev_out)
{
    ENTER(lat);
    NOT_A_SUBSTEP(lat);
    if (!lat->slab) return fail(lat, SU2_ESTATE, "su2_slab_plaquette: not a slab handle");
    if (!dev_out) return fail(lat, SU2_EARG, "su2_slab_plaquette: NULL dev_out");
    if (!lat->initialised) return fail(lat, SU2_ESTATE, "lattice not initialised");
    const double scale = 1.0 / (6.0 * 2.0 * (double)lat->g.st * (double)lat->nt_glob);  // 1 / (6 V_global)
    if (fused)
        lat->launches += launch_final_sum(lat->sc.epart, 3 * heatbath_ctas(lat->g), scale, dev_out, lat->stream);
    else
        lat->launches += launch_plaquette(lat->links, lat->g, lat->precision, lat->sc, dev_out, lat->stream, scale);
    CK(lat, cudaGetLastError());
    return SU2_OK;
}

extern "C" int su2_slab_polyakov(su2_lattice* lat, const void* dev_prev, void* dev_next, double* dev_out)
{
    ENTER(lat);
    NOT_A_SUBSTEP(lat);
    if (!lat->slab) return fail(lat, SU2_ESTATE, "su2_slab_polyakov: not a slab handle");
    if (!lat->initialised) return fail(lat, SU2_ESTATE, "lattice not initialised");
    if ((dev_prev == nullptr) != (lat->t0 == 0))
        return fail(lat, SU2_EARG, "su2_slab_polyakov: dev_prev must be NULL exactly on the slab that holds t = 0");
    if (!dev_next && !dev_out) return fail(lat, SU2_EARG, "su2_slab_polyakov: nothing to write");
    lat->launches += launch_polyakov_chain(lat->links, lat->g, lat->precision, lat->sc, dev_prev, dev_next, dev_out,
                                           lat->stream);
    CK(lat, cudaGetLastError());
    return SU2_OK;
}

// CUDA IPC: lets another process (one per GPU) store into this slab's halos
extern "C" int su2_ipc_export(su2_lattice* lat, void* handle64)
{
    ENTER(lat);
    if (!handle64) return fail(lat, SU2_EARG, "su2_ipc_export: NULL handle buffer");
    if (!lat->owns_links) return fail(lat, SU2_ESTATE, "su2_ipc_export: the links must be library-allocated (su2_slab_create)");
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "cudaIpcMemHandle_t is 64 bytes");
    cudaIpcMemHandle_t h;
    CK(lat, cudaIpcGetMemHandle(&h, lat->links_base));
    memcpy(handle64, &h, sizeof h);
    return SU2_OK;
}

extern "C" int su2_ipc_open(const void* handle64, void** dev_ptr)
{
    if (!handle64 || !dev_ptr) return SU2_EARG;
    cudaIpcMemHandle_t h;
    memcpy(&h, handle64, sizeof h);
    if (cudaIpcOpenMemHandle(dev_ptr, h, cudaIpcMemLazyEnablePeerAccess) != cudaSuccess) {
        cudaGetLastError();
        *dev_ptr = nullptr;
        return SU2_ECUDA;
    }
    return SU2_OK;
}

extern "C" int su2_ipc_close(void* dev_ptr)
{
    if (!dev_ptr) return SU2_OK;
    if (cudaIpcCloseMemHandle(dev_ptr) != cudaSuccess) {
        cudaGetLastError();
        return SU2_ECUDA;
    }
    return SU2_OK;
}

extern "C" int su2_mean_plaquette_noalloc(const void* dev_links, int Nx, int Ny, int Nz, int Nt, int precision,
                                          void* cuda_stream, double* dev_out)
{
    if (!dev_links || !dev_out || ((uintptr_t)dev_links & 31) || !valid_dims(Nx, Ny, Nz, Nt, precision)) return SU2_EARG;
    if ((uint64_t)Nx * Ny * Nz * Nt > SU2_NOALLOC_MAX_SITES) return SU2_ETOOBIG;
    Geom g = {};  // as create_impl fills it for a whole lattice
    g.n[0] = Nx; g.n[1] = Ny; g.n[2] = Nz; g.n[3] = Nt;
    g.nxh = Nx / 2;
    g.sy = g.nxh;
    g.sz = g.nxh * Ny;
    g.st = g.nxh * Ny * Nz;
    g.vh = (uint32_t)((uint64_t)Nx * Ny * Nz * Nt / 2);
    g.wup[0] = -(g.nxh - 1);
    g.wup[1] = -(Ny - 1) * g.sy;
    g.wup[2] = -(Nz - 1) * g.sz;
    g.wup[3] = -(Nt - 1) * g.st;
    g.t_lo = 0;
    g.nt_upd = Nt;
    choose_tiling(g, 1, precision);
    return launch_plaquette_noalloc(dev_links, g, precision, dev_out, (cudaStream_t)cuda_stream);
}

extern "C" int su2_bandwidth_probe(size_t bytes, int passes, int mode, void* cuda_stream, double* gbs_out,
                                   double* us_per_pass_out)
{
    if (!gbs_out || passes < 1 || passes > 100000 || bytes < (1u << 20) || (bytes & 31) ||
        (mode != SU2_PROBE_READ && mode != SU2_PROBE_COPY))
        return SU2_EARG;
    return run_bandwidth_probe(bytes, passes, mode, (cudaStream_t)cuda_stream, gbs_out, us_per_pass_out);
}

extern "C" uint64_t su2_launch_count(const su2_lattice* lat) { return lat ? lat->launches : 0; }

extern "C" void* su2_device_links(su2_lattice* lat) { return lat ? lat->links : nullptr; }

extern "C" const char* su2_last_error(const su2_lattice* lat) { return lat ? lat->msg : "NULL handle"; }

extern "C" const char* su2_strerror(int code)
{
    switch (code) {
        case SU2_OK: return "ok";
        case SU2_EARG: return "bad argument";
        case SU2_EALLOC: return "device allocation failed";
        case SU2_ECUDA: return "CUDA runtime error";
        case SU2_ESTATE: return "bad state: lattice not initialised";
        case SU2_ETOOBIG: return "lattice exceeds SU2_NOALLOC_MAX_SITES, the static scratch of su2_mean_plaquette_noalloc";
        default: return "unknown error code";
    }
}
