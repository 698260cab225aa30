// api.cu -- the C ABI of librosen.so (include/rosen.h): argument validation, per-device scratch,
// host-pointer staging, launches, summary assembly. No compute happens on the host: every step of
// the path runs in the kernels of lattice.cu / realspace.cu / reduce.cu.
#include "../../include/rosen.h"
#include "common.cuh"

#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <vector>

namespace {

using rosen::DevOutputs;
using rosen::Partial;

thread_local char g_err[512] = "";
thread_local int32_t g_launches = 0;
thread_local const char* g_kernel = "";

int fail_cuda(cudaError_t e, const char* what)
{
    std::snprintf(g_err, sizeof(g_err), "%s: %s", what, cudaGetErrorString(e));
    cudaGetLastError();   // clear the sticky-less error state
    return ROSEN_ECUDA;
}
#define CK(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return fail_cuda(e_, #call); } while (0)

// Per-device scratch: block partials + one total, and a pinned host mirror of the total.
struct Scratch;
// RAII: serialises the calls of one device (host side) and orders them across streams (device side).
struct CallGuard {
    Scratch* sc = nullptr; cudaStream_t stream = nullptr;
    int enter(Scratch* s, cudaStream_t st);
    ~CallGuard();
};
struct Scratch {
    Partial*       dev = nullptr;          // [kMaxPartials] block partials
    rosen_summary* summary_dev = nullptr;  // written by finalize_kernel
    uint32_t*      vb_counter = nullptr;   // virtual-block ticket of the lattice kernel
    double*        lmax = nullptr;         // [kMaxPartials + 1] block maxima of lnW and their maximum (long chains)
    rosen_summary* summary_host = nullptr; // pinned mirror
    // long-chain lattice path (lattice_hash.cu): grown on demand, kept until rosen_workspace_release()
    void*          hash_tables = nullptr;  size_t hash_tables_bytes = 0;
    void*          hash_rec = nullptr;     size_t hash_rec_bytes = 0;
    unsigned long long* hash_ticket = nullptr;
    uint32_t*      done_flags = nullptr;   // [kMaxPartials] mapped pinned host memory: virtual blocks whose outputs are stored
    cudaStream_t   copy_stream = nullptr;  // device->host copies of finished conformations while the kernel runs
    uint32_t*      hash_gen = nullptr;     // [kMaxGenSlots] generation counters of the long-chain kernels' threads / warps
    uint64_t       ws_layout = 0;          // signature of the table layout the workspace was last cleared for (0: none)
    double*        perm_thr = nullptr;    // [2][ROSEN_PERM_MAX_N + 1] PERM thresholds (ln_lo | ln_hi)
    // calls of one device share everything above: host threads take call_mutex for the whole call, and a call on another
    // stream than the previous one first waits for that call's last enqueued work (last_done)
    std::mutex     call_mutex;
    cudaEvent_t    last_done = nullptr;
    cudaStream_t   last_stream = nullptr;
    bool           have_last = false;
};
constexpr size_t kHashTableCap = (size_t)12 << 30;  // bytes of per-chain hash tables kept resident at most
constexpr int kMaxDevices = 64;
constexpr size_t kMaxGenSlots = 1 << 20;             // >= resident threads (lattice) / warps (real space) of any device
Scratch g_scratch[kMaxDevices];
std::mutex g_mutex;

int get_scratch(Scratch** out)
{
    int dev = 0;
    CK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) { std::snprintf(g_err, sizeof(g_err), "device index %d unsupported", dev); return ROSEN_ECUDA; }
    std::lock_guard<std::mutex> lock(g_mutex);
    Scratch& s = g_scratch[dev];
    if (!s.dev) {
        // all or nothing: a failed allocation must not leave a half-initialised scratch behind for the next call
        Partial* d = nullptr; rosen_summary* sd = nullptr; uint32_t* vc = nullptr; double* lm = nullptr; rosen_summary* sh = nullptr;
        cudaError_t e = cudaMalloc(&d, sizeof(Partial) * rosen::kMaxPartials);
        if (e == cudaSuccess) e = cudaMalloc(&sd, sizeof(rosen_summary));
        if (e == cudaSuccess) e = cudaMalloc(&vc, sizeof(uint32_t));
        if (e == cudaSuccess) e = cudaMalloc(&lm, sizeof(double) * (rosen::kMaxPartials + 1));
        if (e == cudaSuccess) e = cudaMallocHost(&sh, sizeof(rosen_summary));
        if (e != cudaSuccess) {
            cudaFree(d); cudaFree(sd); cudaFree(vc); cudaFree(lm); if (sh) cudaFreeHost(sh);
            return fail_cuda(e, "per-device scratch allocation");
        }
        s.summary_dev = sd; s.vb_counter = vc; s.lmax = lm; s.summary_host = sh; s.dev = d;
        // host-pointer calls stage through stream-ordered allocations: keep freed staging memory in the pool instead of
        // returning gigabytes to the driver at every synchronisation (config 5: 3.2 GB per call)
        cudaMemPool_t pool = nullptr;
        if (cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess && pool) {
            uint64_t keep = ~0ull;
            cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
        }
        cudaGetLastError();
    }
    *out = &s;
    return ROSEN_OK;
}

int CallGuard::enter(Scratch* s, cudaStream_t st)
{
    s->call_mutex.lock();
    sc = s; stream = st;
    if (!s->last_done) CK(cudaEventCreateWithFlags(&s->last_done, cudaEventDisableTiming));
    // always wait, even when the handle equals the previous call's: a caller may have destroyed that stream with work pending and
    // been handed the same handle value for a new one; waiting on an event of the same stream costs next to nothing
    if (s->have_last) CK(cudaStreamWaitEvent(st, s->last_done, 0));
    return ROSEN_OK;
}
CallGuard::~CallGuard()
{
    if (!sc) return;
    if (sc->last_done && cudaEventRecord(sc->last_done, stream) == cudaSuccess) { sc->last_stream = stream; sc->have_last = true; }
    else cudaGetLastError();
    sc->call_mutex.unlock();
}

int grow(void** ptr, size_t* have, size_t need)
{
    if (*have >= need) return ROSEN_OK;
    if (*ptr) { cudaDeviceSynchronize(); cudaFree(*ptr); *ptr = nullptr; *have = 0; }
    cudaError_t e = cudaMalloc(ptr, need);
    if (e != cudaSuccess) { fail_cuda(e, "cudaMalloc(long-chain workspace)"); *ptr = nullptr; return ROSEN_ENOMEM; }
    *have = need;
    return ROSEN_OK;
}

// Long-chain workspace tables are valid across calls as long as their layout (kernel kind, entries per table, number of
// tables, stride) is the same: every thread / warp keeps its generation counter in hash_gen, so entries of earlier calls
// read as empty. Only a new allocation or a different layout needs the memset (tables and counters to 0).
int prepare_workspace(Scratch* sc, uint64_t layout, size_t table_bytes_total, bool reallocated, cudaStream_t stream)
{
    if (!sc->hash_gen) CK(cudaMalloc(&sc->hash_gen, kMaxGenSlots * sizeof(uint32_t)));
    if (sc->ws_layout != layout || reallocated) {
        CK(cudaMemsetAsync(sc->hash_tables, 0, table_bytes_total, stream));
        CK(cudaMemsetAsync(sc->hash_gen, 0, kMaxGenSlots * sizeof(uint32_t), stream));
        sc->ws_layout = layout;
    }
    return ROSEN_OK;
}

// Host conformation buffers (ROSEN_MEM_HOST + conf): the generation kernel raises a flag in mapped host memory for every
// virtual block whose outputs are stored; this loop copies the finished chain ranges device -> host on a second stream while
// the kernel is still running, so the PCIe transfer of the dump (3.2 GB at config 5) overlaps the generation instead of following it.
int stream_conf_out_loop(Scratch* sc, cudaStream_t gen_stream, const void* conf_dev, void* conf_host, size_t row_bytes,
                    uint64_t n_chains, uint32_t chunk, uint32_t n_vblocks)
{
    volatile uint32_t* flags = sc->done_flags;
    const uint32_t batch = n_vblocks / 32 > 8 ? n_vblocks / 32 : 8;       // virtual blocks per copy: large transfers, ~32 per call
    uint32_t next = 0, seen = 0;
    bool kernel_over = false;
    while (next < n_vblocks) {
        while (seen < n_vblocks && flags[seen] != 0u) ++seen;
        if (seen - next >= batch || (seen == n_vblocks && seen > next) || (kernel_over && seen > next)) {
            const uint64_t c0 = (uint64_t)next * chunk, c1 = (uint64_t)seen * chunk < n_chains ? (uint64_t)seen * chunk : n_chains;
            CK(cudaMemcpyAsync(static_cast<char*>(conf_host) + c0 * row_bytes, static_cast<const char*>(conf_dev) + c0 * row_bytes,
                               (c1 - c0) * row_bytes, cudaMemcpyDeviceToHost, sc->copy_stream));
            next = seen;
            continue;
        }
        if (kernel_over) break;                                           // flags missing although the kernel ended: launch failed
        const cudaError_t q = cudaStreamQuery(gen_stream);
        if (q == cudaSuccess) { kernel_over = true; continue; }           // one more pass over the flags
        if (q != cudaErrorNotReady) return fail_cuda(q, "generation kernel");
    }
    if (next < n_vblocks) { std::snprintf(g_err, sizeof(g_err), "generation kernel ended without storing every virtual block"); return ROSEN_ECUDA; }
    return ROSEN_OK;
}

int stream_conf_out(Scratch* sc, cudaStream_t gen_stream, const void* conf_dev, void* conf_host, size_t row_bytes,
                    uint64_t n_chains, uint32_t chunk, uint32_t n_vblocks)
{
    const int rc = stream_conf_out_loop(sc, gen_stream, conf_dev, conf_host, row_bytes, n_chains, chunk, n_vblocks);
    // on success and on every error path: the copy stream has finished reading the staging buffer before the caller's
    // ~Staging hands it back to the pool on the generation stream
    const cudaError_t e = cudaStreamSynchronize(sc->copy_stream);
    if (rc) { cudaGetLastError(); return rc; }
    if (e != cudaSuccess) return fail_cuda(e, "cudaStreamSynchronize(copy stream)");
    return ROSEN_OK;
}

// Test and tuning knobs, set through rosen_debug_set() (rosen.h) and never read from the environment: a stray variable in
// a user's shell must not change which kernel runs. 0 = the library's default.
std::atomic<int32_t> g_knob_hash_min_n{0}, g_knob_cell_min_n{0}, g_knob_cand_cap{0}, g_knob_hash_blocks_per_sm{0};

// chain length from which the lattice call uses the hash-map kernel: measured crossover with the O(N^2) scan kernel
// (2^24 chains: N = 128 scan 26.8 ms / hash 42.8 ms; N = 256 scan 152 ms / hash 84 ms). The knob lattice_hash_min_n overrides
// it in 2 .. 513 (tests run either kernel over the other's range; decisions do not depend on the choice).
int32_t hash_min_n()
{
    const int32_t v = g_knob_hash_min_n.load();
    return v ? v : ROSEN_LATTICE_HASH_MIN_N;
}

// same for the real-space call (cell-list kernel, realspace_long.cu): measured crossover with the shared-memory scan
// kernel between N = 340 (k = 16) and N = 470 (k = 64); at N = 2048 the cell list is 10x faster. Knob realspace_cell_min_n,
// 2 .. 2049.
int32_t cell_min_n()
{
    const int32_t v = g_knob_cell_min_n.load();
    return v ? v : ROSEN_REALSPACE_CELL_MIN_N;
}

struct Sizes { size_t lnW, alive, m_seq, digest, conf, ree2, rg2; };

Sizes output_sizes(int32_t N, uint64_t n, size_t conf_elem)
{
    Sizes z;
    z.lnW = n * sizeof(double); z.alive = n; z.m_seq = n * (size_t)(N - 1); z.digest = n * sizeof(uint64_t);
    z.conf = n * (size_t)N * 3 * conf_elem; z.ree2 = n * sizeof(double); z.rg2 = n * sizeof(double);
    return z;
}

// Staging of HOST output pointers: device twins allocated on the stream, copied back, freed.
struct Staging {
    DevOutputs dev{};
    bool staged = false;
    cudaStream_t stream = nullptr;
    ~Staging() { release(); }
    void release()
    {
        if (!staged) return;
        void* ptrs[7] = {dev.lnW, dev.alive, dev.m_seq, dev.digest, dev.conf, dev.ree2, dev.rg2};
        for (void* q : ptrs) if (q) cudaFreeAsync(q, stream);
        staged = false;
    }
};

int stage_outputs(const rosen_outputs* o, const Sizes& z, cudaStream_t stream, Staging* st)
{
    st->stream = stream;
    if (!o) return ROSEN_OK;
    if (o->memory == ROSEN_MEM_DEVICE) {
        st->dev = DevOutputs{o->lnW, o->alive, o->m_seq, o->digest, o->conf, o->ree2, o->rg2};
        return ROSEN_OK;
    }
    if (o->memory != ROSEN_MEM_HOST) { std::snprintf(g_err, sizeof(g_err), "outputs->memory must be ROSEN_MEM_DEVICE or ROSEN_MEM_HOST"); return ROSEN_EINVAL; }
    st->staged = true;
    auto alloc = [&](const void* host, size_t bytes, void** d) -> int {
        *d = nullptr;
        if (!host) return ROSEN_OK;
        cudaError_t e = cudaMallocAsync(d, bytes, stream);
        if (e != cudaSuccess) { fail_cuda(e, "cudaMallocAsync(staging)"); return ROSEN_ENOMEM; }
        return ROSEN_OK;
    };
    int rc;
    if ((rc = alloc(o->lnW, z.lnW, (void**)&st->dev.lnW))) return rc;
    if ((rc = alloc(o->alive, z.alive, (void**)&st->dev.alive))) return rc;
    if ((rc = alloc(o->m_seq, z.m_seq, (void**)&st->dev.m_seq))) return rc;
    if ((rc = alloc(o->digest, z.digest, (void**)&st->dev.digest))) return rc;
    if ((rc = alloc(o->conf, z.conf, (void**)&st->dev.conf))) return rc;
    if ((rc = alloc(o->ree2, z.ree2, (void**)&st->dev.ree2))) return rc;
    if ((rc = alloc(o->rg2, z.rg2, (void**)&st->dev.rg2))) return rc;
    return ROSEN_OK;
}

int copy_back(const rosen_outputs* o, const Sizes& z, const Staging& st, cudaStream_t stream, bool conf_done = false)
{
    if (!o || !st.staged) return ROSEN_OK;
    if (o->lnW) CK(cudaMemcpyAsync(o->lnW, st.dev.lnW, z.lnW, cudaMemcpyDeviceToHost, stream));
    if (o->alive) CK(cudaMemcpyAsync(o->alive, st.dev.alive, z.alive, cudaMemcpyDeviceToHost, stream));
    if (o->m_seq) CK(cudaMemcpyAsync(o->m_seq, st.dev.m_seq, z.m_seq, cudaMemcpyDeviceToHost, stream));
    if (o->digest) CK(cudaMemcpyAsync(o->digest, st.dev.digest, z.digest, cudaMemcpyDeviceToHost, stream));
    if (o->conf && !conf_done) CK(cudaMemcpyAsync(o->conf, st.dev.conf, z.conf, cudaMemcpyDeviceToHost, stream));
    if (o->ree2) CK(cudaMemcpyAsync(o->ree2, st.dev.ree2, z.ree2, cudaMemcpyDeviceToHost, stream));
    if (o->rg2) CK(cudaMemcpyAsync(o->rg2, st.dev.rg2, z.rg2, cudaMemcpyDeviceToHost, stream));
    return ROSEN_OK;
}

void derive(rosen_summary* s)
{
    s->mean_ree2 = s->sum_w_ree2 / s->sum_w;
    s->mean_rg2 = s->sum_w_rg2 / s->sum_w;
    s->attrition = (double)s->n_dead / (double)s->n_chains;
    s->ln_mean_W = s->ln_shift + std::log(s->sum_w / (double)s->n_chains);
}

// After the generation kernel: second reduction pass, summary copy, host staging copies, sync.
// summary (host) and summary_dev (device) are both optional; the finalize kernel runs if either is set.
int finish(Scratch* sc, int grid, uint64_t n_chains, double ln_shift, const double* ln_shift_dev, const rosen_outputs* outputs, const Sizes& z,
           Staging& st, rosen_summary* summary, rosen_summary* summary_dev, cudaStream_t stream, bool conf_done = false)
{
    if (summary || summary_dev) {
        rosen_summary* target = summary_dev ? summary_dev : sc->summary_dev;
        if (rosen::launch_finalize(sc->dev, grid, n_chains, ln_shift, ln_shift_dev, target, stream) < 0)
            return fail_cuda(cudaGetLastError(), "finalize_kernel");
        ++g_launches;
        if (summary) CK(cudaMemcpyAsync(sc->summary_host, target, sizeof(rosen_summary), cudaMemcpyDeviceToHost, stream));
    }
    int rc = copy_back(outputs, z, st, stream, conf_done);
    if (rc) return rc;
    st.release();
    if (summary || (outputs && outputs->memory == ROSEN_MEM_HOST)) CK(cudaStreamSynchronize(stream));
    if (summary) *summary = *sc->summary_host;
    return ROSEN_OK;
}

int lattice_impl(int32_t N, uint64_t n_chains, uint64_t seed, uint64_t chain_offset, const rosen_outputs* outputs,
                 rosen_summary* summary, rosen_summary* summary_dev, void* cuda_stream)
{
    g_err[0] = 0; g_launches = 0; g_kernel = "";
    if (N < 2 || n_chains == 0) { std::snprintf(g_err, sizeof(g_err), "need N >= 2 and n_chains >= 1"); return ROSEN_EINVAL; }
    if (N > ROSEN_LATTICE_MAX_N) { std::snprintf(g_err, sizeof(g_err), "lattice N > %d", ROSEN_LATTICE_MAX_N); return ROSEN_ERANGE; }
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    Scratch* sc = nullptr;
    int rc = get_scratch(&sc);
    if (rc) return rc;
    CallGuard guard;
    if ((rc = guard.enter(sc, stream))) return rc;
    const Sizes z = output_sizes(N, n_chains, sizeof(int32_t));
    Staging st;
    if ((rc = stage_outputs(outputs, z, stream, &st))) return rc;

    // nominal shift = the largest possible lnW; for N > 512 the call replaces it by the largest lnW it generated, found on
    // the device before the sums (hp.lmax below, reading A18)
    const double ln_shift = std::log(6.0) + (double)(N - 2) * std::log(5.0);
    if (N >= hash_min_n()) {
        // long chains: per-chain hash map cube -> occupancy bitmap in HBM (lattice_hash.cu)
        rosen::HashParams hp{};
        hp.N = N; hp.n_chains = n_chains; hp.chain_offset = chain_offset;
        hp.key0 = (uint32_t)seed; hp.key1 = (uint32_t)(seed >> 32);
        hp.ln_shift = ln_shift; hp.out = st.dev; hp.partials = sc->dev;
        rosen::partition_chains(n_chains, &hp.chunk, &hp.n_vblocks, 256u);
        hp.entries = rosen::hash_entries(N);
        const size_t table_bytes = (size_t)16 * hp.entries;               // 16-byte entries
        int max_threads = 0;
        if (rosen::hash_max_threads(&max_threads, g_knob_hash_blocks_per_sm.load()) < 0) return fail_cuda(cudaGetLastError(), "device query");
        uint64_t threads = (n_chains + 255) / 256 * 256;
        if (threads > (uint64_t)max_threads) threads = (uint64_t)max_threads;
        const uint64_t by_mem = kHashTableCap / table_bytes / 256 * 256;
        if (threads > by_mem) threads = by_mem;
        {
            std::lock_guard<std::mutex> lock(g_mutex);
            const size_t had = sc->hash_tables_bytes;
            // a smaller or busy GPU: fewer resident tables (results do not depend on how many threads share the chains)
            while ((rc = grow(&sc->hash_tables, &sc->hash_tables_bytes, threads * table_bytes)) == ROSEN_ENOMEM && threads > 256)
                threads = (threads / 2 + 255) / 256 * 256;
            if (rc) return rc;
            if ((rc = grow(&sc->hash_rec, &sc->hash_rec_bytes, n_chains * sizeof(rosen::ChainRecord)))) return rc;
            if (!sc->hash_ticket) CK(cudaMalloc(&sc->hash_ticket, sizeof(unsigned long long)));
            if (threads > kMaxGenSlots) threads = kMaxGenSlots;
            const uint64_t layout = (1ull << 62) | ((uint64_t)hp.entries << 32) | (uint64_t)threads;
            if ((rc = prepare_workspace(sc, layout, threads * table_bytes, sc->hash_tables_bytes != had, stream))) return rc;
        }
        hp.gen_store = sc->hash_gen;
        hp.tables = static_cast<uint64_t*>(sc->hash_tables);
        hp.rec = static_cast<rosen::ChainRecord*>(sc->hash_rec);
        hp.ticket = sc->hash_ticket;
        hp.lmax = N > ROSEN_LATTICE_SCAN_MAX_N ? sc->lmax : nullptr;     // short chains routed here by the env override keep the fixed shift
        CK(cudaMemsetAsync(hp.ticket, 0, sizeof(unsigned long long), stream));
        rc = rosen::launch_lattice_hash(hp, (int)threads, stream, &g_kernel);
        if (rc < 0) return fail_cuda(cudaGetLastError(), "lattice hash kernel launch");
        g_launches += rc;
        return finish(sc, (int)hp.n_vblocks, n_chains, ln_shift, hp.lmax ? hp.lmax + rosen::kMaxPartials : nullptr, outputs, z, st, summary, summary_dev, stream);
    }

    rosen::LatticeParams p{};
    p.N = N; p.n_chains = n_chains; p.chain_offset = chain_offset;
    p.key0 = (uint32_t)seed; p.key1 = (uint32_t)(seed >> 32); p.rk = rosen::philox_round_keys(seed);
    p.ln_shift = ln_shift;
    p.out = st.dev; p.partials = sc->dev; p.vb_counter = sc->vb_counter;
    rosen::partition_chains(n_chains, &p.chunk, &p.n_vblocks);
    CK(cudaMemsetAsync(sc->vb_counter, 0, sizeof(uint32_t), stream));
    int grid = 0;
    rc = rosen::launch_lattice(p, stream, &g_kernel, &grid);
    if (rc < 0) return rc == -2 ? ROSEN_ERANGE : fail_cuda(cudaGetLastError(), "lattice kernel launch");
    g_launches += rc;
    return finish(sc, (int)p.n_vblocks, n_chains, p.ln_shift, nullptr, outputs, z, st, summary, summary_dev, stream);
}

int realspace_impl(int32_t N, uint64_t n_chains, int32_t k_trials, float bond_len, float sigma, uint64_t seed,
                   uint64_t chain_offset, const rosen_outputs* outputs, rosen_summary* summary,
                   rosen_summary* summary_dev, void* cuda_stream)
{
    g_err[0] = 0; g_launches = 0; g_kernel = "";
    if (N < 2 || n_chains == 0 || k_trials < 1 || k_trials > 255 || !(bond_len > 0.0f) || !(sigma >= 0.0f) ||
        !std::isfinite(bond_len) || !std::isfinite(sigma)) {
        std::snprintf(g_err, sizeof(g_err), "need N >= 2, n_chains >= 1, 1 <= k_trials <= 255, bond_len > 0, sigma >= 0 (finite)");
        return ROSEN_EINVAL;
    }
    if (N > ROSEN_REALSPACE_MAX_N) { std::snprintf(g_err, sizeof(g_err), "real-space N > %d", ROSEN_REALSPACE_MAX_N); return ROSEN_ERANGE; }
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    Scratch* sc = nullptr;
    int rc = get_scratch(&sc);
    if (rc) return rc;
    CallGuard guard;
    if ((rc = guard.enter(sc, stream))) return rc;
    const Sizes z = output_sizes(N, n_chains, sizeof(float));
    Staging st;
    if ((rc = stage_outputs(outputs, z, stream, &st))) return rc;

    const float sigma2 = sigma * sigma;         // fp32 product, rounded once
    // conservative candidate radius, rounded up: ((b + sigma)(1 + 2^-9))^2
    const double cand_r = ((double)bond_len + (double)sigma) * (1.0 + 1.0 / 512.0);
    float prefilter2 = (float)(cand_r * cand_r);
    if ((double)prefilter2 < cand_r * cand_r) prefilter2 = std::nextafterf(prefilter2, INFINITY);
    const double ln_shift = (double)(N - 1) * std::log((double)k_trials);

    if (N >= cell_min_n()) {
        // long chains: chain, cell table and cell lists in HBM, one warp per chain (realspace_long.cu)
        rosen::RealLongParams lp{};
        lp.N = N; lp.k = k_trials; lp.n_chains = n_chains; lp.chain_offset = chain_offset;
        lp.key0 = (uint32_t)seed; lp.key1 = (uint32_t)(seed >> 32);
        lp.b = bond_len; lp.sigma2 = sigma2; lp.prefilter2 = prefilter2;
        lp.inv_cell = (float)(1.0 / (cand_r * (1.0 + 1.0 / 64.0)));
        lp.ln_shift = ln_shift; lp.out = st.dev; lp.partials = sc->dev;
        rosen::partition_chains(n_chains, &lp.chunk, &lp.n_vblocks, 256u);
        lp.n_pad = ((uint32_t)N + 7u) & ~7u;
        lp.entries = rosen::hash_entries(N);
        lp.cand_cap = rosen::kRealLongCandCap;
        if (const int32_t v = g_knob_cand_cap.load()) lp.cand_cap = (uint32_t)v;   // test knob: 33 forces the flush path (results do not depend on it)
        lp.warp_bytes = ((uint64_t)lp.n_pad * 16u + (uint64_t)lp.entries * 16u + 255u) & ~(uint64_t)255u;
        int max_warps = 0;
        if (rosen::real_long_max_warps(k_trials, &max_warps) < 0) return fail_cuda(cudaGetLastError(), "device query");
        uint64_t warps = (n_chains + 7) / 8 * 8;
        if (warps > (uint64_t)max_warps) warps = (uint64_t)max_warps;
        const uint64_t by_mem = kHashTableCap / lp.warp_bytes / 8 * 8;
        if (warps > by_mem) warps = by_mem;
        {
            std::lock_guard<std::mutex> lock(g_mutex);
            const size_t had = sc->hash_tables_bytes;
            while ((rc = grow(&sc->hash_tables, &sc->hash_tables_bytes, warps * lp.warp_bytes)) == ROSEN_ENOMEM && warps > 8)
                warps = (warps / 2 + 7) / 8 * 8;
            if (rc) return rc;
            if ((rc = grow(&sc->hash_rec, &sc->hash_rec_bytes, n_chains * sizeof(rosen::ChainRecord)))) return rc;
            if (!sc->hash_ticket) CK(cudaMalloc(&sc->hash_ticket, sizeof(unsigned long long)));
            // the key holds what fixes every table's byte offset: n_pad (where the cell table starts inside a warp's slice), entries and
            // the warp count. The rounded warp_bytes alone would let N = 1000 (n_pad 1000) reuse the tables of N = 1001 (n_pad 1008,
            // same 32256-byte slice), whose chain slots 1000..1007 would then be read as cell entries.
            const uint64_t layout = (2ull << 62) | ((uint64_t)lp.n_pad << 44) | ((uint64_t)lp.entries << 24) | (uint64_t)warps;
            if ((rc = prepare_workspace(sc, layout, warps * lp.warp_bytes, sc->hash_tables_bytes != had, stream))) return rc;
        }
        lp.gen_store = sc->hash_gen;
        lp.work = static_cast<unsigned char*>(sc->hash_tables);
        lp.rec = static_cast<rosen::ChainRecord*>(sc->hash_rec);
        lp.ticket = sc->hash_ticket;
        lp.lmax = N > ROSEN_REALSPACE_SCAN_MAX_N ? sc->lmax : nullptr;   // as in the lattice call
        CK(cudaMemsetAsync(lp.ticket, 0, sizeof(unsigned long long), stream));
        rc = rosen::launch_realspace_long(lp, (int)warps, stream, &g_kernel);
        if (rc < 0) return fail_cuda(cudaGetLastError(), "real-space long-chain kernel launch");
        g_launches += rc;
        return finish(sc, (int)lp.n_vblocks, n_chains, ln_shift, lp.lmax ? lp.lmax + rosen::kMaxPartials : nullptr, outputs, z, st, summary, summary_dev, stream);
    }

    rosen::RealParams p{};
    p.N = N; p.k = k_trials; p.n_chains = n_chains; p.chain_offset = chain_offset;
    p.key0 = (uint32_t)seed; p.key1 = (uint32_t)(seed >> 32);
    p.b = bond_len; p.sigma2 = sigma2; p.prefilter2 = prefilter2;
    p.ln_shift = ln_shift;
    p.out = st.dev; p.partials = sc->dev; p.vb_counter = sc->vb_counter;
    rosen::partition_chains(n_chains, &p.chunk, &p.n_vblocks, 256u);
    CK(cudaMemsetAsync(sc->vb_counter, 0, sizeof(uint32_t), stream));
    // large dump into host memory: stream the finished conformations out while the kernel runs
    const bool overlap = st.staged && outputs->conf != nullptr && p.n_vblocks >= 64;
    if (overlap) {
        std::lock_guard<std::mutex> lock(g_mutex);
        if (!sc->done_flags) CK(cudaHostAlloc(reinterpret_cast<void**>(&sc->done_flags), rosen::kMaxPartials * sizeof(uint32_t), cudaHostAllocMapped));
        if (!sc->copy_stream) CK(cudaStreamCreateWithFlags(&sc->copy_stream, cudaStreamNonBlocking));
    }
    if (overlap) {
        CK(cudaStreamSynchronize(stream));                               // staging buffers exist before the copy stream reads them
        std::memset(sc->done_flags, 0, p.n_vblocks * sizeof(uint32_t));
        uint32_t* dflags = nullptr;
        CK(cudaHostGetDevicePointer(reinterpret_cast<void**>(&dflags), sc->done_flags, 0));
        p.done = dflags;
    }
    int grid = 0;
    rc = rosen::launch_realspace(p, stream, &g_kernel, &grid);
    if (rc < 0) return rc == -2 ? ROSEN_ERANGE : fail_cuda(cudaGetLastError(), "real-space kernel launch");
    g_launches += rc;
    if (overlap && (rc = stream_conf_out(sc, stream, st.dev.conf, outputs->conf, (size_t)N * 3 * sizeof(float), n_chains, p.chunk, p.n_vblocks)))
        return rc;
    return finish(sc, (int)p.n_vblocks, n_chains, p.ln_shift, nullptr, outputs, z, st, summary, summary_dev, stream, overlap);
}

// Fixed-point Boltzmann factors of the model calls: Q[c] = round(p_c 2^16), p_0 = 1, p_c = p_{c-1} q in fp64.
void model_table(double beta_eps, uint64_t Q[32])
{
    const double q = std::exp(beta_eps);
    double pw = 1.0;
    for (int c = 0; c < 32; ++c) { Q[c] = (uint64_t)std::llround(pw * 65536.0); pw *= q; }
}

int lattice_model_impl(int32_t N, uint64_t n_chains, uint64_t seed, uint64_t chain_offset, int32_t z, double beta_eps,
                       const rosen_outputs* outputs, rosen_summary* summary, void* cuda_stream)
{
    g_err[0] = 0; g_launches = 0; g_kernel = "";
    if (N < 2 || n_chains == 0 || (z != 6 && z != 26) || !(beta_eps >= 0.0) || !(beta_eps <= ROSEN_MODEL_MAX_BETA_EPS)) {
        std::snprintf(g_err, sizeof(g_err), "need N >= 2, n_chains >= 1, z = 6 or 26, 0 <= beta_eps <= %.2f", ROSEN_MODEL_MAX_BETA_EPS);
        return ROSEN_EINVAL;
    }
    if (N > ROSEN_LATTICE_MODEL_MAX_N) { std::snprintf(g_err, sizeof(g_err), "lattice model N > %d", ROSEN_LATTICE_MODEL_MAX_N); return ROSEN_ERANGE; }
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    Scratch* sc = nullptr;
    int rc = get_scratch(&sc);
    if (rc) return rc;
    CallGuard guard;
    if ((rc = guard.enter(sc, stream))) return rc;
    const Sizes zs = output_sizes(N, n_chains, sizeof(int32_t));
    Staging st;
    if ((rc = stage_outputs(outputs, zs, stream, &st))) return rc;
    rosen::ModelParams mp{};
    mp.N = N; mp.z = z; mp.n_chains = n_chains; mp.chain_offset = chain_offset;
    mp.key0 = (uint32_t)seed; mp.key1 = (uint32_t)(seed >> 32);
    model_table(beta_eps, mp.Q);
    mp.out = st.dev; mp.partials = sc->dev;
    rosen::partition_chains(n_chains, &mp.chunk, &mp.n_vblocks, 256u);
    {
        std::lock_guard<std::mutex> lock(g_mutex);
        if ((rc = grow(&sc->hash_rec, &sc->hash_rec_bytes, n_chains * sizeof(rosen::ChainRecord)))) return rc;
    }
    mp.rec = static_cast<rosen::ChainRecord*>(sc->hash_rec);
    mp.lmax = sc->lmax;
    rc = rosen::launch_lattice_model(mp, stream, &g_kernel);
    if (rc < 0) return fail_cuda(cudaGetLastError(), "lattice model kernel launch");
    g_launches += rc;
    return finish(sc, (int)mp.n_vblocks, n_chains, 0.0, mp.lmax + rosen::kMaxPartials, outputs, zs, st, summary, nullptr, stream);
}

int realspace_model_impl(int32_t N, uint64_t n_chains, int32_t k_trials, float bond_len, float sigma, float lambda, double beta_eps,
                         uint64_t seed, uint64_t chain_offset, const rosen_outputs* outputs, rosen_summary* summary, void* cuda_stream)
{
    g_err[0] = 0; g_launches = 0; g_kernel = "";
    if (N < 2 || n_chains == 0 || k_trials < 1 || k_trials > 255 || !(bond_len > 0.0f) || !(sigma >= 0.0f) ||
        !std::isfinite(bond_len) || !std::isfinite(sigma) || !(lambda >= 1.0f) || !std::isfinite(lambda) ||
        !(beta_eps >= 0.0) || !(beta_eps <= ROSEN_MODEL_MAX_BETA_EPS)) {
        std::snprintf(g_err, sizeof(g_err), "need N >= 2, n_chains >= 1, 1 <= k_trials <= 255, bond_len > 0, sigma >= 0, lambda >= 1 (finite), 0 <= beta_eps <= %.2f",
                      ROSEN_MODEL_MAX_BETA_EPS);
        return ROSEN_EINVAL;
    }
    if (N > ROSEN_REALSPACE_MODEL_MAX_N) { std::snprintf(g_err, sizeof(g_err), "real-space model N > %d", ROSEN_REALSPACE_MODEL_MAX_N); return ROSEN_ERANGE; }
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    Scratch* sc = nullptr;
    int rc = get_scratch(&sc);
    if (rc) return rc;
    CallGuard guard;
    if ((rc = guard.enter(sc, stream))) return rc;
    const Sizes zs = output_sizes(N, n_chains, sizeof(float));
    Staging st;
    if ((rc = stage_outputs(outputs, zs, stream, &st))) return rc;
    const float well = lambda * sigma;              // fp32 products, rounded once each
    rosen::RealParams p{};
    p.N = N; p.k = k_trials; p.n_chains = n_chains; p.chain_offset = chain_offset;
    p.key0 = (uint32_t)seed; p.key1 = (uint32_t)(seed >> 32);
    p.b = bond_len; p.sigma2 = sigma * sigma; p.well2 = well * well;
    // conservative candidate radius around the well instead of the core: ((b + lambda sigma)(1 + 2^-9))^2, rounded up
    const double cand_r = ((double)bond_len + (double)well) * (1.0 + 1.0 / 512.0);
    p.prefilter2 = (float)(cand_r * cand_r);
    if ((double)p.prefilter2 < cand_r * cand_r) p.prefilter2 = std::nextafterf(p.prefilter2, INFINITY);
    p.ln_shift = 0.0;
    model_table(beta_eps, p.Q);
    p.out = st.dev; p.partials = sc->dev; p.vb_counter = sc->vb_counter;
    rosen::partition_chains(n_chains, &p.chunk, &p.n_vblocks, 256u);
    {
        std::lock_guard<std::mutex> lock(g_mutex);
        if ((rc = grow(&sc->hash_rec, &sc->hash_rec_bytes, n_chains * sizeof(rosen::ChainRecord)))) return rc;
    }
    p.rec = static_cast<rosen::ChainRecord*>(sc->hash_rec);
    CK(cudaMemsetAsync(sc->vb_counter, 0, sizeof(uint32_t), stream));
    int grid = 0;
    rc = rosen::launch_realspace(p, stream, &g_kernel, &grid);
    if (rc < 0) return rc == -2 ? ROSEN_ERANGE : fail_cuda(cudaGetLastError(), "real-space model kernel launch");
    g_launches += rc;
    rc = rosen::launch_reduce_records(p.rec, n_chains, p.chunk, p.n_vblocks, 0.0, sc->lmax, st.dev, sc->dev, stream);
    if (rc < 0) return fail_cuda(cudaGetLastError(), "record reduction");
    g_launches += rc;
    return finish(sc, (int)p.n_vblocks, n_chains, 0.0, sc->lmax + rosen::kMaxPartials, outputs, zs, st, summary, nullptr, stream);
}

int perm_impl(int32_t N, uint64_t n_tours, uint64_t seed, uint64_t tour_offset, const double* ln_lo, const double* ln_hi,
              double ln_ref, uint32_t max_nodes, const rosen_outputs* outputs, rosen_summary* summary, void* cuda_stream)
{
    g_err[0] = 0; g_launches = 0; g_kernel = "";
    if (N < 2 || n_tours == 0 || !ln_lo || !ln_hi || max_nodes == 0 || !std::isfinite(ln_ref) ||
        (outputs && (outputs->m_seq || outputs->conf))) {
        std::snprintf(g_err, sizeof(g_err), "need N >= 2, n_tours >= 1, thresholds, max_nodes >= 1, finite ln_ref; per-tour outputs are lnW, alive, digest, ree2, rg2");
        return ROSEN_EINVAL;
    }
    for (int32_t n = 2; n < N && n <= ROSEN_PERM_MAX_N; ++n)
        if (std::isnan(ln_lo[n]) || std::isnan(ln_hi[n])) { std::snprintf(g_err, sizeof(g_err), "NaN threshold at length %d", n); return ROSEN_EINVAL; }
    if (N > ROSEN_PERM_MAX_N) { std::snprintf(g_err, sizeof(g_err), "PERM N > %d", ROSEN_PERM_MAX_N); return ROSEN_ERANGE; }
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    Scratch* sc = nullptr;
    int rc = get_scratch(&sc);
    if (rc) return rc;
    CallGuard guard;
    if ((rc = guard.enter(sc, stream))) return rc;
    const Sizes zs = output_sizes(N, n_tours, sizeof(int32_t));
    Staging st;
    if ((rc = stage_outputs(outputs, zs, stream, &st))) return rc;
    {
        std::lock_guard<std::mutex> lock(g_mutex);
        if ((rc = grow(&sc->hash_rec, &sc->hash_rec_bytes, n_tours * sizeof(rosen::ChainRecord)))) return rc;
        if (!sc->hash_ticket) CK(cudaMalloc(&sc->hash_ticket, sizeof(unsigned long long)));
        if (!sc->perm_thr) CK(cudaMalloc(&sc->perm_thr, sizeof(double) * 2 * (ROSEN_PERM_MAX_N + 1)));
    }
    CK(cudaMemcpyAsync(sc->perm_thr, ln_lo, sizeof(double) * (size_t)(N + 1), cudaMemcpyHostToDevice, stream));
    CK(cudaMemcpyAsync(sc->perm_thr + ROSEN_PERM_MAX_N + 1, ln_hi, sizeof(double) * (size_t)(N + 1), cudaMemcpyHostToDevice, stream));
    CK(cudaMemsetAsync(sc->hash_ticket, 0, sizeof(unsigned long long), stream));
    rosen::PermParams pp{};
    pp.N = N; pp.n_tours = n_tours; pp.tour_offset = tour_offset;
    pp.key0 = (uint32_t)seed; pp.key1 = (uint32_t)(seed >> 32);
    pp.ln_lo = sc->perm_thr; pp.ln_hi = sc->perm_thr + ROSEN_PERM_MAX_N + 1; pp.ln_ref = ln_ref; pp.max_nodes = max_nodes;
    pp.out = st.dev; pp.partials = sc->dev;
    rosen::partition_chains(n_tours, &pp.chunk, &pp.n_vblocks, 256u);
    pp.rec = static_cast<rosen::ChainRecord*>(sc->hash_rec);
    pp.lmax = sc->lmax; pp.ticket = sc->hash_ticket;
    rc = rosen::launch_lattice_perm(pp, stream, &g_kernel);
    if (rc < 0) return fail_cuda(cudaGetLastError(), "PERM kernel launch");
    g_launches += rc;
    return finish(sc, (int)pp.n_vblocks, n_tours, 0.0, pp.lmax + rosen::kMaxPartials, outputs, zs, st, summary, nullptr, stream);
}

// ---- rosen_lattice_generate_noalloc: the lattice scan kernel with its scratch in static device memory ----------------
// For callers that may not allocate (rosen.h says who and why). Nothing below calls cudaMalloc*, cudaFree*, cudaHostAlloc,
// or creates a stream or an event, and it does not touch the Scratch of the other entry points (get_scratch allocates).
//
// Layout of the array: [0, kNoAllocPartialBytes) block partials, one per virtual block; then the 4-byte virtual-block
// ticket in a 256-byte slot of its own, so that the memset of the ticket never shares a line with a partial.
constexpr size_t kNoAllocPartialBytes = sizeof(Partial) * rosen::kMaxPartials;
static_assert(kNoAllocPartialBytes + 256 == ROSEN_NOALLOC_SCRATCH_BYTES, "rosen.h states the size of the static scratch");
static_assert(ROSEN_NOALLOC_MAX_CHAINS == (uint64_t)rosen::kMaxPartials * rosen::kMinChunk, "one partial per kMinChunk chains");
static __device__ __align__(256) unsigned char g_noalloc_scratch[ROSEN_NOALLOC_SCRATCH_BYTES];

// In host code `g_noalloc_scratch` is only a handle for the runtime's symbol table, NOT a device address: handing it to a
// kernel would fault (or, on a machine where the GPU can read host memory, quietly use the wrong memory). The address is
// asked for once per device, with that device current, and cached here.
unsigned char* g_noalloc_addr[kMaxDevices] = {};
std::mutex g_noalloc_mutex;

int noalloc_scratch(unsigned char** out)
{
    int dev = 0;
    CK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) { std::snprintf(g_err, sizeof(g_err), "device index %d unsupported", dev); return ROSEN_ECUDA; }
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_addr[dev]) {
        void* addr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&addr, g_noalloc_scratch);
        if (e != cudaSuccess || !addr) return fail_cuda(e != cudaSuccess ? e : cudaErrorInvalidSymbol, "cudaGetSymbolAddress(static scratch)");
        g_noalloc_addr[dev] = static_cast<unsigned char*>(addr);
    }
    *out = g_noalloc_addr[dev];
    return ROSEN_OK;
}

int lattice_noalloc_impl(int32_t N, uint64_t n_chains, uint64_t seed, uint64_t chain_offset, const rosen_outputs* outputs,
                         rosen_summary* summary_dev, void* cuda_stream)
{
    g_err[0] = 0; g_launches = 0; g_kernel = "";
    if (N < 2 || n_chains == 0) { std::snprintf(g_err, sizeof(g_err), "need N >= 2 and n_chains >= 1"); return ROSEN_EINVAL; }
    if (outputs && outputs->memory != ROSEN_MEM_DEVICE) {
        std::snprintf(g_err, sizeof(g_err), "rosen_lattice_generate_noalloc takes device outputs only (a host destination needs a staging allocation)");
        return ROSEN_EINVAL;
    }
    if (N > ROSEN_NOALLOC_MAX_N) {
        std::snprintf(g_err, sizeof(g_err), "rosen_lattice_generate_noalloc: N = %d exceeds ROSEN_NOALLOC_MAX_N = %d (longer chains need the "
                      "allocating rosen_lattice_generate)", N, ROSEN_NOALLOC_MAX_N);
        return ROSEN_ERANGE;
    }
    if (n_chains > ROSEN_NOALLOC_MAX_CHAINS) {
        std::snprintf(g_err, sizeof(g_err), "rosen_lattice_generate_noalloc: n_chains = %llu exceeds ROSEN_NOALLOC_MAX_CHAINS = %llu, the capacity of the "
                      "static scratch (split the range over several calls with chain_offset)",
                      (unsigned long long)n_chains, (unsigned long long)ROSEN_NOALLOC_MAX_CHAINS);
        return ROSEN_ERANGE;
    }
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    unsigned char* scratch = nullptr;
    int rc = noalloc_scratch(&scratch);
    if (rc) return rc;

    rosen::LatticeParams p{};
    p.N = N; p.n_chains = n_chains; p.chain_offset = chain_offset;
    p.key0 = (uint32_t)seed; p.key1 = (uint32_t)(seed >> 32); p.rk = rosen::philox_round_keys(seed);
    p.ln_shift = std::log(6.0) + (double)(N - 2) * std::log(5.0);
    if (outputs) p.out = DevOutputs{outputs->lnW, outputs->alive, outputs->m_seq, outputs->digest, outputs->conf, outputs->ree2, outputs->rg2};
    p.partials = reinterpret_cast<Partial*>(scratch);
    p.vb_counter = reinterpret_cast<uint32_t*>(scratch + kNoAllocPartialBytes);
    rosen::partition_chains(n_chains, &p.chunk, &p.n_vblocks);          // the regular call's partition: same sums, bit for bit
    if (p.n_vblocks > (uint32_t)rosen::kMaxPartials) { std::snprintf(g_err, sizeof(g_err), "static scratch too small for %u virtual blocks", p.n_vblocks); return ROSEN_ERANGE; }
    // the array keeps whatever the last call left: the ticket must start at 0; partials [0, n_vblocks) are all rewritten by
    // the kernel before the second pass reads them, the rest is never read
    CK(cudaMemsetAsync(p.vb_counter, 0, sizeof(uint32_t), stream));
    int grid = 0;
    rc = rosen::launch_lattice(p, stream, &g_kernel, &grid);
    if (rc < 0) return rc == -2 ? ROSEN_ERANGE : fail_cuda(cudaGetLastError(), "lattice kernel launch");
    g_launches += rc;
    if (summary_dev) {
        if (rosen::launch_finalize(p.partials, (int)p.n_vblocks, n_chains, p.ln_shift, nullptr, summary_dev, stream) < 0)
            return fail_cuda(cudaGetLastError(), "finalize_kernel");
        ++g_launches;
    }
    return ROSEN_OK;
}

}  // namespace

extern "C" {

int rosen_lattice_generate(int32_t N, uint64_t n_chains, uint64_t seed, uint64_t chain_offset,
                           const rosen_outputs* outputs, rosen_summary* summary, void* cuda_stream)
{
    return lattice_impl(N, n_chains, seed, chain_offset, outputs, summary, nullptr, cuda_stream);
}

int rosen_realspace_generate(int32_t N, uint64_t n_chains, int32_t k_trials, float bond_len, float sigma,
                             uint64_t seed, uint64_t chain_offset,
                             const rosen_outputs* outputs, rosen_summary* summary, void* cuda_stream)
{
    return realspace_impl(N, n_chains, k_trials, bond_len, sigma, seed, chain_offset, outputs, summary, nullptr, cuda_stream);
}

int rosen_lattice_generate_async(int32_t N, uint64_t n_chains, uint64_t seed, uint64_t chain_offset,
                                 const rosen_outputs* outputs, rosen_summary* summary_device, void* cuda_stream)
{
    if (outputs && outputs->memory != ROSEN_MEM_DEVICE) {
        std::snprintf(g_err, sizeof(g_err), "the _async calls take device outputs only"); return ROSEN_EINVAL;
    }
    return lattice_impl(N, n_chains, seed, chain_offset, outputs, nullptr, summary_device, cuda_stream);
}

int rosen_realspace_generate_async(int32_t N, uint64_t n_chains, int32_t k_trials, float bond_len, float sigma,
                                   uint64_t seed, uint64_t chain_offset,
                                   const rosen_outputs* outputs, rosen_summary* summary_device, void* cuda_stream)
{
    if (outputs && outputs->memory != ROSEN_MEM_DEVICE) {
        std::snprintf(g_err, sizeof(g_err), "the _async calls take device outputs only"); return ROSEN_EINVAL;
    }
    return realspace_impl(N, n_chains, k_trials, bond_len, sigma, seed, chain_offset, outputs, nullptr, summary_device, cuda_stream);
}

int rosen_lattice_generate_noalloc(int32_t N, uint64_t n_chains, uint64_t seed, uint64_t chain_offset,
                                   const rosen_outputs* outputs, rosen_summary* summary_device, void* cuda_stream)
{
    return lattice_noalloc_impl(N, n_chains, seed, chain_offset, outputs, summary_device, cuda_stream);
}

int rosen_lattice_dump(int32_t N, uint64_t n_chains, uint64_t seed, uint64_t chain_offset,
                       int32_t* conf, double* lnW, int32_t memory, rosen_summary* summary, void* cuda_stream)
{
    rosen_outputs o{};
    o.conf = conf; o.lnW = lnW; o.memory = memory;
    return rosen_lattice_generate(N, n_chains, seed, chain_offset, &o, summary, cuda_stream);
}

int rosen_realspace_dump(int32_t N, uint64_t n_chains, int32_t k_trials, float bond_len, float sigma,
                         uint64_t seed, uint64_t chain_offset,
                         float* conf, double* lnW, int32_t memory, rosen_summary* summary, void* cuda_stream)
{
    rosen_outputs o{};
    o.conf = conf; o.lnW = lnW; o.memory = memory;
    return rosen_realspace_generate(N, n_chains, k_trials, bond_len, sigma, seed, chain_offset, &o, summary, cuda_stream);
}

int rosen_lattice_generate_model(int32_t N, uint64_t n_chains, uint64_t seed, uint64_t chain_offset, int32_t z, double beta_eps,
                                 const rosen_outputs* outputs, rosen_summary* summary, void* cuda_stream)
{
    return lattice_model_impl(N, n_chains, seed, chain_offset, z, beta_eps, outputs, summary, cuda_stream);
}

int rosen_realspace_generate_model(int32_t N, uint64_t n_chains, int32_t k_trials, float bond_len, float sigma, float lambda,
                                   double beta_eps, uint64_t seed, uint64_t chain_offset,
                                   const rosen_outputs* outputs, rosen_summary* summary, void* cuda_stream)
{
    return realspace_model_impl(N, n_chains, k_trials, bond_len, sigma, lambda, beta_eps, seed, chain_offset, outputs, summary, cuda_stream);
}

int rosen_lattice_perm(int32_t N, uint64_t n_tours, uint64_t seed, uint64_t tour_offset, const double* ln_lo, const double* ln_hi,
                       double ln_ref, uint32_t max_nodes, const rosen_outputs* outputs, rosen_summary* summary, void* cuda_stream)
{
    return perm_impl(N, n_tours, seed, tour_offset, ln_lo, ln_hi, ln_ref, max_nodes, outputs, summary, cuda_stream);
}

int rosen_summary_merge(const rosen_summary* parts, int32_t count, rosen_summary* merged)
{
    if (!parts || !merged || count < 1) return ROSEN_EINVAL;
    // common shift = the largest of the parts' (equal for short chains; per-call maxima for long chains, reading A18):
    // sums are rescaled by exp(L_i - L) (squared for sum_w2), a factor of exactly 1 when the shifts agree
    for (int32_t i = 0; i < count; ++i)
        if (!std::isfinite(parts[i].ln_shift)) return ROSEN_EINVAL;
    double L = parts[0].ln_shift;
    bool have = parts[0].sum_w > 0.0;
    for (int32_t i = 1; i < count; ++i)
        if (parts[i].sum_w > 0.0 && (!have || parts[i].ln_shift > L)) { L = parts[i].ln_shift; have = true; }
    rosen_summary m{};
    m.ln_shift = L;
    for (int32_t i = 0; i < count; ++i) {
        const rosen_summary& q = parts[i];
        const double f = q.sum_w > 0.0 ? std::exp(q.ln_shift - L) : 0.0;
        m.n_chains += q.n_chains; m.n_dead += q.n_dead; m.n_steps_attempted += q.n_steps_attempted;
        m.sum_w += f * q.sum_w; m.sum_w_ree2 += f * q.sum_w_ree2; m.sum_w_rg2 += f * q.sum_w_rg2; m.sum_w2 += f * f * q.sum_w2;
        m.digest_xor ^= q.digest_xor; m.digest_sum += q.digest_sum;
    }
    derive(&m);
    *merged = m;
    return ROSEN_OK;
}

int rosen_fit_exponents(const int32_t* N, const double* mean_ree2, const double* ln_mean_W,
                        int32_t count, int32_t use_steps, rosen_fit* fit)
{
    if (!N || !mean_ree2 || !ln_mean_W || !fit || count < 2) return ROSEN_EINVAL;
    const double nan = std::nan("");
    // normal equations of y = p0 + p1 x + p2 lx  (Eq. 7) and of r = q0 + q1 lx (Eq. 4), centred for conditioning
    double mx = 0, ml = 0, my = 0, mr = 0;
    for (int32_t i = 0; i < count; ++i) {
        if (N[i] < 2 || !(mean_ree2[i] > 0.0) || !std::isfinite(mean_ree2[i]) || !std::isfinite(ln_mean_W[i])) return ROSEN_EINVAL;
        const double x = (double)(N[i] - (use_steps ? 1 : 0));
        mx += x; ml += std::log(x); my += ln_mean_W[i]; mr += std::log(mean_ree2[i]);
    }
    mx /= count; ml /= count; my /= count; mr /= count;
    double sxx = 0, sxl = 0, sll = 0, sxy = 0, sly = 0, slr = 0;
    for (int32_t i = 0; i < count; ++i) {
        const double x = (double)(N[i] - (use_steps ? 1 : 0));
        const double dx = x - mx, dl = std::log(x) - ml, dy = ln_mean_W[i] - my, dr = std::log(mean_ree2[i]) - mr;
        sxx += dx * dx; sxl += dx * dl; sll += dl * dl; sxy += dx * dy; sly += dl * dy; slr += dl * dr;
    }
    if (!(sll > 0.0)) return ROSEN_EINVAL;
    rosen_fit f;
    const double slope = slr / sll;
    f.nu = 0.5 * slope; f.ln_a = mr - slope * ml;
    f.mu = f.gamma = f.c = f.rms_lnZ = nan;
    double p1 = 0, p2 = 0;
    if (count >= 3) {
        const double det = sxx * sll - sxl * sxl;
        if (!(std::fabs(det) > 1e-14 * sxx * sll)) return ROSEN_EINVAL;
        p1 = (sxy * sll - sly * sxl) / det; p2 = (sly * sxx - sxy * sxl) / det;
        f.mu = std::exp(p1); f.gamma = p2 + 1.0; f.c = my - p1 * mx - p2 * ml;
    }
    double e1 = 0, e2 = 0;
    for (int32_t i = 0; i < count; ++i) {
        const double x = (double)(N[i] - (use_steps ? 1 : 0)), lx = std::log(x);
        const double r1 = std::log(mean_ree2[i]) - (f.ln_a + slope * lx); e1 += r1 * r1;
        if (count >= 3) { const double r2 = ln_mean_W[i] - (f.c + p1 * x + p2 * lx); e2 += r2 * r2; }
    }
    f.rms_ree2 = std::sqrt(e1 / count);
    if (count >= 3) f.rms_lnZ = std::sqrt(e2 / count);
    *fit = f;
    return ROSEN_OK;
}

int rosen_realspace_dump_probe(int32_t N, uint64_t n_chains, float* conf, double* lnW, void* cuda_stream)
{
    g_err[0] = 0; g_launches = 0; g_kernel = "dump_probe_kernel<G=32>";
    if (N < 2 || N > ROSEN_REALSPACE_SCAN_MAX_N || n_chains == 0 || !conf) {
        std::snprintf(g_err, sizeof(g_err), "need 2 <= N <= %d, n_chains >= 1 and a device conf buffer", ROSEN_REALSPACE_SCAN_MAX_N);
        return ROSEN_EINVAL;
    }
    if (rosen::launch_dump_probe(N, n_chains, conf, lnW, static_cast<cudaStream_t>(cuda_stream)) < 0)
        return fail_cuda(cudaGetLastError(), "dump_probe_kernel");
    g_launches = 1;
    return ROSEN_OK;
}

int rosen_direction_eval(const uint32_t* wz, const uint32_t* wphi, uint64_t n, float* dir_xyz, int32_t memory, void* cuda_stream)
{
    g_err[0] = 0; g_launches = 0; g_kernel = "direction_eval_kernel";
    if (!wz || !wphi || !dir_xyz || n == 0 || (memory != ROSEN_MEM_DEVICE && memory != ROSEN_MEM_HOST)) {
        std::snprintf(g_err, sizeof(g_err), "need wz, wphi, dir_xyz, n >= 1 and a valid memory kind"); return ROSEN_EINVAL;
    }
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    if (memory == ROSEN_MEM_DEVICE) {
        if (rosen::launch_direction_eval(wz, wphi, n, dir_xyz, stream) < 0) return fail_cuda(cudaGetLastError(), "direction_eval_kernel");
        ++g_launches;
        return ROSEN_OK;
    }
    uint32_t *dz = nullptr, *dp = nullptr; float* dout = nullptr;
    cudaError_t e = cudaMallocAsync((void**)&dz, n * 4, stream);
    if (e == cudaSuccess) e = cudaMallocAsync((void**)&dp, n * 4, stream);
    if (e == cudaSuccess) e = cudaMallocAsync((void**)&dout, n * 12, stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(dz, wz, n * 4, cudaMemcpyHostToDevice, stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(dp, wphi, n * 4, cudaMemcpyHostToDevice, stream);
    if (e == cudaSuccess && rosen::launch_direction_eval(dz, dp, n, dout, stream) < 0) e = cudaGetLastError();
    if (e == cudaSuccess) { ++g_launches; e = cudaMemcpyAsync(dir_xyz, dout, n * 12, cudaMemcpyDeviceToHost, stream); }
    if (dz) cudaFreeAsync(dz, stream);
    if (dp) cudaFreeAsync(dp, stream);
    if (dout) cudaFreeAsync(dout, stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
    return e == cudaSuccess ? ROSEN_OK : fail_cuda(e, "rosen_direction_eval");
}

size_t rosen_workspace_bytes(void)
{
    size_t b = sizeof(Partial) * rosen::kMaxPartials + sizeof(rosen_summary);
    int dev = 0;
    if (cudaGetDevice(&dev) == cudaSuccess && dev >= 0 && dev < kMaxDevices) {
        std::lock_guard<std::mutex> lock(g_mutex);
        const Scratch& s = g_scratch[dev];
        b += s.hash_tables_bytes + s.hash_rec_bytes;
        if (s.hash_gen) b += kMaxGenSlots * sizeof(uint32_t);
        if (s.perm_thr) b += sizeof(double) * 2 * (ROSEN_PERM_MAX_N + 1);
    } else {
        cudaGetLastError();
    }
    return b;
}

int rosen_workspace_release(void)
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) { cudaGetLastError(); return ROSEN_OK; }   // nothing was ever allocated
    Scratch& s = g_scratch[dev];
    // call_mutex first, then g_mutex: the order the generate calls use. A call of another host thread that has already read
    // the workspace pointers into its kernel parameters finishes enqueueing before anything is freed; the device
    // synchronisation below then waits for that work.
    std::lock_guard<std::mutex> call_lock(s.call_mutex);
    std::lock_guard<std::mutex> lock(g_mutex);
    if (s.dev) cudaDeviceSynchronize();                 // s.dev: some call has used this device
    if (s.hash_tables) { cudaFree(s.hash_tables); s.hash_tables = nullptr; s.hash_tables_bytes = 0; }
    if (s.hash_gen) { cudaFree(s.hash_gen); s.hash_gen = nullptr; }
    s.ws_layout = 0;
    if (s.hash_rec) { cudaFree(s.hash_rec); s.hash_rec = nullptr; s.hash_rec_bytes = 0; }
    if (s.hash_ticket) { cudaFree(s.hash_ticket); s.hash_ticket = nullptr; }
    if (s.perm_thr) { cudaFree(s.perm_thr); s.perm_thr = nullptr; }
    // what the host-dump overlap and the cross-stream ordering created on demand; the next call that needs them makes them again
    if (s.done_flags) { cudaFreeHost(s.done_flags); s.done_flags = nullptr; }
    if (s.copy_stream) { cudaStreamDestroy(s.copy_stream); s.copy_stream = nullptr; }
    if (s.last_done) { cudaEventDestroy(s.last_done); s.last_done = nullptr; }
    s.have_last = false; s.last_stream = nullptr;       // the device is idle: nothing left to order against
    // staging memory of host-pointer calls stays in the device's default memory pool (get_scratch raises its release
    // threshold so that gigabytes are not returned to the driver at every synchronisation): hand the unused part back now
    if (s.dev) {
        cudaMemPool_t pool = nullptr;
        if (cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess && pool) cudaMemPoolTrimTo(pool, 0);
    }
    cudaGetLastError();
    return ROSEN_OK;
}
int rosen_debug_set(const char* knob, int64_t value)
{
    g_err[0] = 0;
    if (!knob) { std::snprintf(g_err, sizeof(g_err), "rosen_debug_set: knob is NULL"); return ROSEN_EINVAL; }
    auto set = [&](std::atomic<int32_t>& k, int64_t lo, int64_t hi) -> int {
        if (value != 0 && (value < lo || value > hi)) {
            std::snprintf(g_err, sizeof(g_err), "rosen_debug_set(%s): %lld outside %lld .. %lld (0 = default)", knob, (long long)value, (long long)lo, (long long)hi);
            return ROSEN_EINVAL;
        }
        k.store((int32_t)value);
        return ROSEN_OK;
    };
    if (!std::strcmp(knob, "lattice_hash_min_n")) return set(g_knob_hash_min_n, 2, ROSEN_LATTICE_SCAN_MAX_N + 1);
    if (!std::strcmp(knob, "realspace_cell_min_n")) return set(g_knob_cell_min_n, 2, ROSEN_REALSPACE_SCAN_MAX_N + 1);
    if (!std::strcmp(knob, "realspace_cand_cap")) return set(g_knob_cand_cap, 33, (int64_t)rosen::kRealLongCandCap);
    if (!std::strcmp(knob, "hash_blocks_per_sm")) return set(g_knob_hash_blocks_per_sm, 1, 32);
    if (!std::strcmp(knob, "generations_left")) {
        // every generation counter of the current device's long-chain workspace := (largest generation of the kernel the
        // workspace was last laid out for) - value, so that each thread / warp clears its table and restarts at
        // generation 1 after `value` more chains: the only way a test reaches that branch (2^25 / 2^19 chains per thread otherwise)
        int dev = 0;
        CK(cudaGetDevice(&dev));
        if (dev < 0 || dev >= kMaxDevices) return ROSEN_EINVAL;
        Scratch& sc = g_scratch[dev];
        std::lock_guard<std::mutex> call_lock(sc.call_mutex);
        std::lock_guard<std::mutex> lock(g_mutex);
        const uint64_t kind = sc.ws_layout >> 62;
        if (!sc.hash_gen || (kind != 1 && kind != 2)) {
            std::snprintf(g_err, sizeof(g_err), "rosen_debug_set(generations_left): no long-chain workspace on this device yet");
            return ROSEN_EINVAL;
        }
        const uint32_t gen_max = kind == 1 ? rosen::lattice_hash_gen_max() : rosen::real_long_gen_max();
        if (value < 0 || value > (int64_t)gen_max) { std::snprintf(g_err, sizeof(g_err), "rosen_debug_set(generations_left): 0 .. %u", gen_max); return ROSEN_EINVAL; }
        CK(cudaDeviceSynchronize());
        // the tables are cleared too: entries of earlier calls may carry the very generations the preset counters are about
        // to run through again, which never happens when the counters only count up
        CK(cudaMemset(sc.hash_tables, 0, sc.hash_tables_bytes));
        const std::vector<uint32_t> host(kMaxGenSlots, gen_max - (uint32_t)value);
        CK(cudaMemcpy(sc.hash_gen, host.data(), kMaxGenSlots * sizeof(uint32_t), cudaMemcpyHostToDevice));
        return ROSEN_OK;
    }
    std::snprintf(g_err, sizeof(g_err), "rosen_debug_set: unknown knob '%s'", knob);
    return ROSEN_EINVAL;
}

int32_t rosen_last_launch_count(void) { return g_launches; }
const char* rosen_last_kernel_name(void) { return g_kernel; }

const char* rosen_strerror(int code)
{
    switch (code) {
        case ROSEN_OK: return "success";
        case ROSEN_EINVAL: return "invalid argument";
        case ROSEN_ERANGE: return "chain length beyond the supported range";
        case ROSEN_ECUDA: return "CUDA runtime error";
        case ROSEN_ENOMEM: return "device allocation failed";
        default: return "unknown error code";
    }
}
const char* rosen_last_error(void) { return g_err; }
const char* rosen_version(void) { return "rosen-b200 0.1 (sm_100a)"; }

}  // extern "C"
