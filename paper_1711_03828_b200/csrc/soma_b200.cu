// soma_b200.cu -- C ABI (include/soma_b200.h) and host-side orchestration of the SCMF step.
//
// Device memory layout:
//   x, y, z     three fp32 arrays, chain-major; every architecture's segment starts on a 512-byte
//               boundary (128 floats) so that a warp tile of the fused kernel is 3 x LDG.128 per lane
//   omega, counts   two formats (soma_ctx::pack, SOMA_OPT_COUNT_BITS):
//               planes   float32 omega[n_types][cells], uint32 counts[n_types][cells]
//               records  (two types) omega[cells] = {omega_A, omega_B}; counts uint32 [cells], n_A in the low and
//                        n_B in the high 16 bits (PAPER.md:243 stores uint16; overflow is detected by the field
//                        kernel, SOMA_EOVERFLOW): 12 instead of 16 bytes per cell, the default once the planes
//                        would not stay in L2.  The C ABI's [type][cell] arrays: export_grid_kernel (soma_fields)
//   toff        uint32 per monomer of every architecture: the offset of its type in omega (type * cells, or type)
//   decisions   1 bit per bead (only written with SOMA_OPT_RECORD_DECISIONS)
//   acc_slots   256 spread 64-bit counters of accepted moves
//   orig        uint32 per chain slot: the caller's index of the chain stored there (soma_layout.cuh);
//               chains are kept in Hilbert order of their centres of mass (SOMA_OPT_LAYOUT), re-sorted
//               every SOMA_OPT_SORT_INTERVAL sweeps
#include "soma_kernels.cuh"
#include "soma_layout.cuh"

#include <cub/device/device_radix_sort.cuh>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/soma_b200.h"

namespace {

thread_local std::string g_err;

int fail(int code, const char* fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_err = buf;
    return code;
}

#define CU(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess)                                                                     \
            return fail(e_ == cudaErrorMemoryAllocation ? SOMA_ENOMEM : SOMA_ECUDA, "%s: %s (%s:%d)", \
                        #call, cudaGetErrorString(e_), __FILE__, __LINE__);                        \
    } while (0)

// Every entry point works on the device its context was created on, whatever device is current in the
// calling thread, and leaves the caller's current device as it found it.
struct DeviceGuard {
    int prev = -1, want = -1;
    explicit DeviceGuard(int device) : want(device)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        if (prev != want) cudaSetDevice(want);
    }
    ~DeviceGuard()
    {
        if (prev >= 0 && prev != want) cudaSetDevice(prev);
    }
};

struct Spec {
    uint64_t n_chains = 0;
    uint32_t N = 0;
    uint64_t n_beads = 0;   // n_chains * N
    uint64_t local0 = 0;    // index of the architecture's first bead in the caller's arrays (= gid0 unless sharded)
    uint64_t gid0 = 0;      // global index of the first bead (unpadded, the API's bead index)
    uint64_t off = 0;       // offset of the segment in the padded device arrays
    uint32_t toff_off = 0;  // offset into the toff table
    bool fused_ok = false;  // 4 | N, N <= 128
    bool any_n = false;     // fused_ok and N does not divide 128: floor(128 / N) chains per tile, idle lanes (kAnyN)
    uint32_t log2N = 0;     // fused_ok: log2 N, or (any_n) the chains per tile
    uint64_t chain_off = 0; // offset into orig[]
    uint32_t n_tiles = 0;   // full 128-bead tiles (fused_ok only)
    // general architecture (bond list): the device words of Fig. 2 and the set members behind them at arch_off
    bool general = false;
    uint32_t n_bonds = 0;
    uint64_t arch_off = 0;
    std::vector<uint32_t> set_off;   // [n_sets + 1] offsets into members[]
    uint32_t n_arch_words = 0;       // Fig. 2 words | members | set_off | set_magic
    // grid and shared memory of the fused kernel in random set order (launch_fused), kept per instantiation asked last
    mutable const void* order_kernel = nullptr;
    mutable int order_device = -1, order_blocks = 0;
    mutable size_t order_smem = 0;
};

constexpr int kEventPool = 2048;
constexpr int kMaxDevices = 64;

}  // namespace

struct soma_ctx {
    std::vector<Spec> specs;
    int n_types = 0, N_ref = 0;
    float box[3] = {0, 0, 0};
    int grid[3] = {0, 0, 0};
    float chiN[soma::kMaxTypes][soma::kMaxTypes] = {};
    float kappaN = 0, A = 0;
    uint64_t seed = 0;
    uint64_t n_beads = 0, n_pad = 0, cells = 0;
    uint64_t n_beads_global = 0;     // beads of the whole system (= n_beads unless this context is a shard)
    int sharded = 0;                 // created by soma_init_shard: soma_shard_moves / soma_shard_fields instead of soma_step
    // peer mode (soma_shard_set_peers): the field kernel reduces the ranks' exchange arrays itself over peer memory.
    // The allocation holds two buffers of n_types * cells words used alternately (exchange = the current one).
    uint32_t* exchange_base = nullptr;
    int n_peers = 0, my_rank = 0, peer_parity = 0;
    std::vector<void*> peer_opened;          // CUDA IPC mappings to close
    const uint32_t** peer_table = nullptr;   // device: [n_peers] base addresses of the ranks' allocations
    uint32_t* exchange = nullptr;    // shard: what this rank's move kernels count into; summed over the ranks by the caller,
                                     // folded into counts (the whole system's numbers) by the field kernel, which clears it
    bool counts_pending = false;     // shard: counts was cleared by a histogram (which went into the exchange array) and is
                                     // not the whole system's numbers until the next soma_shard_fields folds the sum in

    float *x = nullptr, *y = nullptr, *z = nullptr;
    uint32_t* counts = nullptr;      // planes [n_types][cells], or packed [cells] (pack)
    float* omega = nullptr;          // planes [n_types][cells], or records [cells][2] (pack)
    int count_bits = 0;              // SOMA_OPT_COUNT_BITS: 0 auto, 16, 32
    bool pack = false;               // occupation numbers of two types packed 16 + 16 bits per cell
    unsigned long long* ticket_sum = nullptr;   // device: ticket and sum of the field kernel's overflow check
    uint32_t* overflow_host = nullptr;   // pinned, mapped: sticky flag the kernels set (a packed half overflowed)
    uint32_t* overflow_dev = nullptr;    // its device address
    void* grid_stage = nullptr;      // [n_types][cells] floats + uint32: soma_fields to host memory (allocated on first use)
    uint32_t* toff = nullptr;        // per monomer of every architecture: type * cells (planes) or type (records)
    std::vector<uint32_t> types_host;    // the bead types behind toff
    uint32_t* arch = nullptr;        // architectures given by bond lists (Spec::arch_off)
    float* ext = nullptr;            // [n_types][cells] static external field, or null
    uint8_t* forbidden = nullptr;    // [cells] 1 = no particle may enter, or null
    uint64_t n_forbidden = 0;
    uint32_t* decisions = nullptr;
    unsigned long long* acc_slots = nullptr;
    unsigned long long* acc_host = nullptr;  // pinned staging for soma_stats

    // layout (soma_layout.cuh)
    uint32_t* orig = nullptr;        // [n_chains of all architectures]
    uint32_t* orig_tmp = nullptr;
    float* scratch = nullptr;        // n_pad floats: target of a permutation, then swapped in
    float* stage = nullptr;          // 3 * n_beads floats in the caller's order (allocated on first use)
    uint32_t *sort_keys[2] = {nullptr, nullptr}, *sort_vals[2] = {nullptr, nullptr};
    void* cub_tmp = nullptr;
    size_t cub_tmp_bytes = 0;
    uint64_t n_chains_total = 0, max_chains = 0;
    int layout = 1;                  // 0: caller's order, 1: Hilbert order
    int scheme = 0;                  // 0: independent sets (Code 2); 1: molecule-parallel random picks (Code 1, R24)
    int set_order = 0;               // 0: even set then odd set; 1: random per chain and sweep (R21)
    int field_interval = 1;          // omega refreshed after every field_interval-th sweep (R22)
    int sort_interval = 2000;        // sweeps between re-sorts (0: only at init / set_positions)
    uint64_t sweeps_since_sort = 0;

    cudaStream_t stream = nullptr;
    int device = 0, n_sm = 0;

    // options
    int hamiltonian = 0, move = 1, record = 0, kernel_choice = 0, density_mode = 0, timing = 0;
    uint32_t* n_outside = nullptr;   // device counter: beads whose coordinates are outside the supported domain
    int pdl = 1;             // programmatic dependent launch of the fused and field kernels (SOMA_OPT_PDL)
    float smc_step = 0.0f;

    uint64_t sweep = 0, attempted = 0, launches = 0;
    bool decisions_valid = false;

    // timing
    std::vector<cudaEvent_t> ev;   // pairs
    std::vector<int> ev_class;
    int ev_used = 0;
    double t_ms[SOMA_K_COUNT] = {};
    uint64_t t_launches[SOMA_K_COUNT] = {};

    soma::GridP gridp() const;
    soma::MoveP movep(uint64_t sweep_no) const;
    soma::FieldP fieldp() const;
};

soma::GridP soma_ctx::gridp() const
{
    soma::GridP g;
    for (int a = 0; a < 3; ++a) {
        g.inv_L[a] = (float)(1.0 / (double)box[a]);
        g.nf[a] = (float)grid[a];
        g.n[a] = (uint32_t)grid[a];
        g.neg_n[a] = 0u - (uint32_t)grid[a];
    }
    const uint32_t Mb = 0x4B400000u;   // bits of 1.5 * 2^23
    const uint32_t Kx = (g.n[0] - 1u) * Mb, Ky = (g.n[1] - 1u) * Mb, Kz = (g.n[2] - 1u) * Mb;
    g.k_rec = ((Kx * g.n[1] + Ky) * g.n[2] + Kz) * (pack ? 2u : 1u);
    g.cells = (uint32_t)cells;
    g.last = (uint32_t)(cells * (size_t)n_types) - 1u;
    return g;
}

soma::MoveP soma_ctx::movep(uint64_t sweep_no) const
{
    soma::MoveP p;
    p.g = gridp();
    p.c1 = (float)(2.0 * (double)A);
    p.c0 = (float)((double)A * (std::ldexp(1.0, -23) - 3.0));
    p.hk = (float)(1.5 * ((double)N_ref - 1.0));
    p.k0 = (float)(3.0 * ((double)N_ref - 1.0));
    p.a_s = smc_step;
    p.noise = sqrtf(2.0f * smc_step);
    p.four_as = 4.0f * smc_step;
    for (uint32_t r = 0; r < 10; ++r) {
        p.rk[r][0] = (uint32_t)seed + r * 0x9E3779B9u;
        p.rk[r][1] = (uint32_t)(seed >> 32) + r * 0xBB67AE85u;
    }
    p.sweep_lo = (uint32_t)sweep_no;
    p.sweep_hi = (uint32_t)(sweep_no >> 32);
    // Philox rounds 1-2 over the counter words every bead shares (philox4x32_10_head)
    for (uint32_t sub = 0; sub < 2; ++sub) {
        const uint32_t tag = ((uint32_t)move << 8) | sub;
        const uint64_t pc1 = (uint64_t)p.sweep_hi * 0xCD9E8D57ull;
        const uint32_t a1 = (uint32_t)(pc1 >> 32) ^ p.sweep_lo ^ p.rk[0][0];
        const uint64_t pa2 = (uint64_t)a1 * 0xD2511F53ull;
        p.head[sub][0] = tag ^ p.rk[0][1];
        p.head[sub][1] = (uint32_t)pc1 ^ p.rk[1][0];
        p.head[sub][2] = (uint32_t)(pa2 >> 32) ^ p.rk[1][1];
        p.head[sub][3] = (uint32_t)pa2;
    }
    return p;
}

soma::FieldP soma_ctx::fieldp() const
{
    soma::FieldP f;
    f.inv_nbar = (float)((double)(cells - n_forbidden) / (double)n_beads_global);   // accessible volume (R23)
    f.kappa0 = (float)((double)kappaN / (double)N_ref);
    for (int i = 0; i < soma::kMaxTypes; ++i)
        for (int k = 0; k < soma::kMaxTypes; ++k) {
            f.chi0[i][k] = (float)((double)chiN[i][k] / (double)N_ref);
            f.half_chi0[i][k] = (float)(0.5 * (double)chiN[i][k] / (double)N_ref);
        }
    f.n_types = n_types;
    f.hamiltonian = hamiltonian;
    f.cells = (uint32_t)cells;
    return f;
}

namespace {

// ---- kernel timing (SOMA_OPT_TIMING) ------------------------------------------------------------
int drain_events(soma_ctx* c)
{
    if (c->ev_used == 0) return SOMA_OK;
    CU(cudaStreamSynchronize(c->stream));
    for (int i = 0; i < c->ev_used; ++i) {
        float ms = 0.f;
        CU(cudaEventElapsedTime(&ms, c->ev[2 * i], c->ev[2 * i + 1]));
        c->t_ms[c->ev_class[i]] += ms;
    }
    c->ev_used = 0;
    return SOMA_OK;
}

struct Timed {
    soma_ctx* c;
    int slot = -1;
    Timed(soma_ctx* ctx, int klass, int n_launches) : c(ctx)
    {
        c->launches += n_launches;
        if (!c->timing) return;
        if (c->ev.empty()) {
            c->ev.resize(2 * kEventPool);
            c->ev_class.resize(kEventPool);
            for (auto& e : c->ev) cudaEventCreate(&e);
        }
        if (c->ev_used == kEventPool) drain_events(c);
        slot = c->ev_used++;
        c->ev_class[slot] = klass;
        c->t_launches[klass] += n_launches;
        cudaEventRecord(c->ev[2 * slot], c->stream);
    }
    ~Timed()
    {
        if (slot >= 0) cudaEventRecord(c->ev[2 * slot + 1], c->stream);
    }
};

// ---- architecture of a molecule type given by its bond list ----------------------------------------
// Appends to `words` the array of Fig. 2 (layout in soma_kernels.cuh): N | per monomer (index of
// its first bond word << 8 | type) | per bond (signed partner offset << 5 | bond type << 1 | last-bond flag), and
// behind it the independent sets (greedy first fit in monomer order, R25): members[N] (set by set) |
// set_off[n_sets + 1] | set_magic[n_sets].  Indices are relative to the first word appended.  Host only.
int build_architecture(const soma_chain_spec& spec, int a, std::vector<uint32_t>& words, std::vector<uint32_t>& set_off)
{
    const uint32_t N = spec.n_beads, n_bonds = spec.n_bonds;
    if (!spec.bonds) return fail(SOMA_EINVAL, "soma_init: spec %d: n_bonds > 0 but bonds is NULL", a);
    // neighbour lists in ascending order
    std::vector<std::vector<uint32_t>> nb(N);
    for (uint32_t b = 0; b < n_bonds; ++b) {
        const uint32_t i = spec.bonds[2 * b], j = spec.bonds[2 * b + 1];
        if (i >= N || j >= N || i == j)
            return fail(SOMA_EINVAL, "soma_init: spec %d bond %u (%u, %u): need i != j, both < n_beads", a, b, i, j);
        nb[i].push_back(j);
        nb[j].push_back(i);
    }
    std::vector<uint32_t> set_of(N, 0);
    uint32_t n_sets = 0;
    for (uint32_t j = 0; j < N; ++j) {
        std::sort(nb[j].begin(), nb[j].end());
        if (std::adjacent_find(nb[j].begin(), nb[j].end()) != nb[j].end())
            return fail(SOMA_EINVAL, "soma_init: spec %d: a bond of monomer %u is listed twice", a, j);
        uint32_t col = 0;
        for (bool clash = true; clash; ) {
            clash = false;
            for (uint32_t k : nb[j]) if (k < j && set_of[k] == col) clash = true;
            if (clash) ++col;
        }
        set_of[j] = col;
        n_sets = std::max(n_sets, col + 1);
    }
    if (1 + (uint64_t)N + 2 * (uint64_t)n_bonds >= (1u << 24) || N >= (1u << 26))
        return fail(SOMA_EINVAL, "soma_init: spec %d: architecture too large for the 24-bit bond-list offsets of Fig. 2", a);
    const size_t first = words.size();
    words.push_back(N);
    uint32_t run = 1 + N;
    for (uint32_t j = 0; j < N; ++j) {
        words.push_back(((nb[j].empty() ? 0u : run) << 8) | (spec.types ? spec.types[j] : 0u));
        run += (uint32_t)nb[j].size();
    }
    for (uint32_t j = 0; j < N; ++j)
        for (size_t q = 0; q < nb[j].size(); ++q)
            words.push_back(((uint32_t)((int32_t)nb[j][q] - (int32_t)j) << 5) | (q + 1 == nb[j].size() ? 1u : 0u));
    set_off.assign(1, 0);
    for (uint32_t col = 0; col < n_sets; ++col) {
        for (uint32_t j = 0; j < N; ++j) if (set_of[j] == col) words.push_back(j);
        set_off.push_back((uint32_t)(words.size() - first - (1 + N) - 2 * (size_t)n_bonds));
    }
    // for the staged kernel: division by the set size as a multiply
    for (uint32_t v : set_off) words.push_back(v);
    for (uint32_t col = 0; col < n_sets; ++col)
        words.push_back((uint32_t)((1ull << 32) / (set_off[col + 1] - set_off[col])) + 1u);
    return SOMA_OK;
}

// ---- launches -----------------------------------------------------------------------------------
// where the move and histogram kernels count: a shard counts its contribution into the exchange array
inline uint32_t* count_target(const soma_ctx* c) { return c->sharded ? c->exchange : c->counts; }

bool spec_uses_fused(const soma_ctx* c, const Spec& s)
{
    if (c->kernel_choice == 1) return false;
    if (c->move == 2 && c->set_order == 1) return false;   // Smart-MC in random set order: generic kernel only
    if (!s.fused_ok) return false;
    return true;
}

// Launch with the programmatic-serialization attribute (programmatic dependent launch): the kernel may
// become resident while its predecessor in the stream drains; it calls soma::pdl_wait() before it
// touches anything the predecessor writes.  pdl = 0 (SOMA_OPT_PDL): an ordinary launch.
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(bool pdl, void (*kernel)(KArgs...), unsigned blocks, unsigned threads, size_t smem,
                       cudaStream_t stream, Args&&... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(blocks);
    cfg.blockDim = dim3(threads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

template <int kMove, bool kIncr, bool kRecord, bool kOrder, bool kPack, bool kAnyN>
int launch_fused(soma_ctx* c, const soma::MoveP& P, const Spec& s)
{
    auto kernel = soma::fused_sweep_kernel<kMove, kIncr, kRecord, kOrder, kPack, kAnyN>;
    constexpr int threads = soma::kFusedThreads, warps_per_block = threads / 32;
    // blocks per SM of this instantiation (without dynamic shared memory) and the shared memory a block may ask for,
    // asked once per device; the mutex makes the first launches of two threads safe
    static std::mutex mu;
    static int resident[kMaxDevices] = {};
    static size_t smem_limit[kMaxDevices] = {};
    const int dev_slot = c->device % kMaxDevices;
    {
        std::lock_guard<std::mutex> lock(mu);
        if (resident[dev_slot] == 0) {
            int r = 0;
            if (kOrder) {
                // shared memory for the order bits of a block's chains: 160 KB, or what the device grants a block if
                // that is less (static shared memory of the kernel taken off)
                int optin = 0;
                cudaFuncAttributes fa;
                CU(cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, c->device));
                CU(cudaFuncGetAttributes(&fa, kernel));
                size_t lim = std::min<size_t>(160 * 1024, (size_t)optin > fa.sharedSizeBytes ? (size_t)optin - fa.sharedSizeBytes : 0);
                if (lim < 1024) return fail(SOMA_ECUDA, "launch_fused: the device grants a block %d bytes of shared memory", optin);
                CU(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)lim));
                smem_limit[dev_slot] = lim;
            }
            CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&r, kernel, threads, 0));
            resident[dev_slot] = r < 1 ? 1 : r;
        }
    }
    const int res = resident[dev_slot];
    int per_sm = res;                                  // every block resident, one wave
    int blocks = c->n_sm * per_sm;
    const int max_useful = (int)((s.n_tiles + warps_per_block - 1) / warps_per_block);
    if (blocks > max_useful) blocks = max_useful;
    // random set order: four bytes per chain of the longest tile range a block can get (the chains grouped by
    // their order bit); more (not all resident) blocks if that does not fit into shared memory.  The shared memory
    // may lower the number of resident blocks, and fewer blocks need more of it each: iterate to the fixed point
    // (per_sm only falls; on a B200 the kernel's registers allow one block per SM and the loop runs once).  The
    // result depends on the spec and the instantiation only: kept with the spec.
    size_t order_smem = 0;
    if (kOrder) {
        if (s.order_kernel == (const void*)kernel && s.order_device == c->device) {
            blocks = s.order_blocks;
            order_smem = s.order_smem;
        } else {
            const size_t limit = smem_limit[dev_slot];
            const size_t chains_per_tile = soma::kTile / s.N;      // floor: also for kAnyN
            for (;;) {
                for (int waves = 1;; ++waves) {
                    blocks = std::min(c->n_sm * per_sm * waves, max_useful);
                    order_smem = ((size_t)s.n_tiles / blocks + 1) * chains_per_tile * 4 + 16;
                    if (order_smem <= limit || blocks == max_useful) break;
                }
                if (order_smem > limit) return fail(SOMA_ECUDA, "launch_fused: order bits of one warp's tiles exceed shared memory");
                int r = 0;
                CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&r, kernel, threads, order_smem));
                if (r < 1) r = 1;
                if (r >= per_sm) break;
                per_sm = r;
            }
            s.order_kernel = (const void*)kernel;
            s.order_device = c->device;
            s.order_blocks = blocks;
            s.order_smem = order_smem;
        }
    }
    Timed t(c, SOMA_K_MOVE, 1);
    CU(launch_pdl(c->pdl != 0, kernel, (unsigned)blocks, (unsigned)threads, order_smem, c->stream,
                  P, c->x + s.off, c->y + s.off, c->z + s.off, c->omega, count_target(c), c->toff + s.toff_off,
                  kAnyN ? s.N : s.N - 1u, s.n_tiles, (uint32_t)s.gid0, c->orig + s.chain_off, s.log2N, c->decisions,
                  c->acc_slots));
    return SOMA_OK;
}

template <int kMove, bool kIncr, bool kRecord, bool kPack>
int launch_moves_t(soma_ctx* c, const soma::MoveP& P)
{
    for (const Spec& s : c->specs) {
        if (s.n_beads == 0) continue;
        if (s.general) {        // bond-list architecture: the independent sets one after the other
            const uint32_t* arch = c->arch + s.arch_off;
            const uint32_t* members = arch + 1 + s.N + 2 * (size_t)s.n_bonds;
            // molecules staged in shared memory, every set in one launch (positions cross HBM once per sweep)
            const uint32_t group = std::max<uint32_t>(1u, 256u / s.N);   // ~256 beads per warp and pass (measured: 219 us at C3 against 232 with 512, 292 with 1024)
            const int warps = 8;
            const size_t head = ((size_t)s.n_arch_words + s.N + 3) & ~(size_t)3;
            const size_t smem = sizeof(uint32_t) * head + sizeof(float) * 3 * (size_t)warps * group * s.N;
            if (c->kernel_choice != 1 && (size_t)group * s.N <= 65535 && smem <= 200 * 1024) {
                auto kernel = soma::arch_staged_kernel<kMove, kIncr, kRecord, kPack>;
                static size_t asked_smem[kMaxDevices] = {};
                static int asked_res[kMaxDevices] = {};
                const int d = c->device % kMaxDevices;
                if (asked_smem[d] != smem) {
                    if (smem > 48 * 1024) CU(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
                    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&asked_res[d], kernel, warps * 32, smem));
                    if (asked_res[d] < 1) asked_res[d] = 1;
                    asked_smem[d] = smem;
                }
                const uint64_t n_groups = (s.n_chains + group - 1) / group;
                const uint64_t blocks = std::min<uint64_t>((uint64_t)c->n_sm * asked_res[d], (n_groups + warps - 1) / warps);
                Timed t(c, SOMA_K_MOVE, 1);
                kernel<<<(unsigned)blocks, warps * 32, smem, c->stream>>>(
                    P, c->x + s.off, c->y + s.off, c->z + s.off, c->omega, count_target(c), c->toff + s.toff_off, arch,
                    s.n_arch_words, s.N, s.n_bonds, (uint32_t)(s.set_off.size() - 1), group, s.n_chains, (uint32_t)s.gid0,
                    c->orig + s.chain_off, c->decisions, c->acc_slots);
                CU(cudaGetLastError());
                continue;
            }
            for (size_t i_set = 0; i_set + 1 < s.set_off.size(); ++i_set) {
                const uint32_t set_size = s.set_off[i_set + 1] - s.set_off[i_set];
                const uint64_t n_items = s.n_chains * set_size;
                const int threads = 256;
                Timed t(c, SOMA_K_MOVE, 1);
                soma::arch_move_kernel<kMove, kIncr, kRecord, kPack><<<(unsigned)((n_items + threads - 1) / threads), threads, 0, c->stream>>>(
                    P, c->x + s.off, c->y + s.off, c->z + s.off, c->omega, count_target(c), c->toff + s.toff_off, arch,
                    members + s.set_off[i_set], s.N, set_size, n_items, (uint32_t)s.gid0, c->orig + s.chain_off,
                    c->decisions, c->acc_slots);
            }
            CU(cudaGetLastError());
            continue;
        }
        if (c->scheme == 1) {   // Code 1: one thread per molecule
            const size_t per_warp = sizeof(float) * 96 * (size_t)s.N;     // 32 chains x 3 coordinates
            const int warps = (int)std::min<size_t>(4, (200 * 1024) / per_warp);
            if (warps >= 1 && c->kernel_choice != 1) {   // chains staged in shared memory
                auto kernel = soma::molecule_staged_kernel<kMove, kIncr, kRecord, kPack>;
                const size_t smem = per_warp * warps;
                // shared-memory limit and resident blocks per SM: asked once per (instantiation, device, chain length)
                static size_t asked_smem[kMaxDevices] = {};
                static int asked_res[kMaxDevices] = {};
                const int d = c->device % kMaxDevices;
                if (asked_smem[d] != smem) {
                    if (smem > 48 * 1024) CU(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
                    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&asked_res[d], kernel, warps * 32, smem));
                    if (asked_res[d] < 1) asked_res[d] = 1;
                    asked_smem[d] = smem;
                }
                const int per_sm = asked_res[d];
                const uint64_t n_groups = (s.n_chains + 31) / 32;
                const uint64_t blocks = std::min<uint64_t>((uint64_t)c->n_sm * per_sm, (n_groups + warps - 1) / warps);
                Timed t(c, SOMA_K_MOVE, 1);
                kernel<<<(unsigned)blocks, warps * 32, smem, c->stream>>>(
                    P, c->x + s.off, c->y + s.off, c->z + s.off, c->omega, count_target(c), c->toff + s.toff_off, s.N,
                    s.n_chains, (uint32_t)s.gid0, c->orig + s.chain_off, c->decisions, c->acc_slots);
                CU(cudaGetLastError());
                continue;
            }
            const int threads = 128;
            const unsigned blocks = (unsigned)((s.n_chains + threads - 1) / threads);
            Timed t(c, SOMA_K_MOVE, 1);
            soma::molecule_move_kernel<kMove, kIncr, kRecord, kPack><<<blocks, threads, 0, c->stream>>>(
                P, c->x + s.off, c->y + s.off, c->z + s.off, c->omega, count_target(c), c->toff + s.toff_off, s.N,
                s.n_chains, (uint32_t)s.gid0, c->orig + s.chain_off, c->decisions, c->acc_slots);
            CU(cudaGetLastError());
            continue;
        }
        float *x = c->x + s.off, *y = c->y + s.off, *z = c->z + s.off;
        const uint32_t* toff = c->toff + s.toff_off;
        uint64_t done = 0;   // beads of this architecture handled by the fused kernel
        if (spec_uses_fused(c, s) && s.n_tiles > 0) {
            const bool order = kMove == 1 && c->set_order == 1;
            int rc = s.any_n ? (order ? launch_fused<kMove, kIncr, kRecord, kMove == 1, kPack, true>(c, P, s)
                                      : launch_fused<kMove, kIncr, kRecord, false, kPack, true>(c, P, s))
                             : (order ? launch_fused<kMove, kIncr, kRecord, kMove == 1, kPack, false>(c, P, s)
                                      : launch_fused<kMove, kIncr, kRecord, false, kPack, false>(c, P, s));
            if (rc) return rc;
            done = s.any_n ? (uint64_t)s.n_tiles * s.log2N * s.N : (uint64_t)s.n_tiles * soma::kTile;
        }
        if (done < s.n_beads) {   // whole chains the fused kernel does not cover (all of them, or a ragged tail)
            const uint64_t n_chains = (s.n_beads - done) / s.N;
            for (uint32_t parity = 0; parity < 2; ++parity) {
                const uint32_t half = (s.N + 1) / 2;
                const uint64_t n_items = n_chains * half;
                const int threads = 256;
                const uint64_t blocks = (n_items + threads - 1) / threads;
                Timed t(c, SOMA_K_MOVE, 1);
                soma::generic_move_kernel<kMove, kIncr, kRecord, kPack><<<(unsigned)blocks, threads, 0, c->stream>>>(
                    P, x + done, y + done, z + done, c->omega, count_target(c), toff, s.N, half, parity,
                    (uint32_t)c->set_order, n_items,
                    (uint32_t)s.gid0, c->orig + s.chain_off + done / s.N, c->decisions, c->acc_slots);
            }
        }
        CU(cudaGetLastError());
    }
    return SOMA_OK;
}

template <int kMove, bool kIncr, bool kRecord>
int launch_moves_3(soma_ctx* c, const soma::MoveP& P)
{
    return c->pack ? launch_moves_t<kMove, kIncr, kRecord, true>(c, P) : launch_moves_t<kMove, kIncr, kRecord, false>(c, P);
}
template <int kMove, bool kIncr>
int launch_moves_2(soma_ctx* c, const soma::MoveP& P)
{
    return c->record ? launch_moves_3<kMove, kIncr, true>(c, P) : launch_moves_3<kMove, kIncr, false>(c, P);
}
template <int kMove>
int launch_moves_1(soma_ctx* c, const soma::MoveP& P)
{
    return c->density_mode == 0 ? launch_moves_2<kMove, true>(c, P) : launch_moves_2<kMove, false>(c, P);
}
int launch_moves(soma_ctx* c, const soma::MoveP& P)
{
    return c->move == 2 ? launch_moves_1<2>(c, P) : launch_moves_1<1>(c, P);
}

// Which grid format SOMA_OPT_COUNT_BITS asks for.  Auto (0): records with packed counters for two bead types
// once the planes (16 bytes per cell) would take more than kPackAutoBytes -- measured on a B200 (126 MB L2):
// C3 (8 MB of planes) 100.3 us per step with planes, 104.3 with records (the packed update costs ~20
// instructions per 128 moves in an issue-bound kernel); C4 (131 MB) 1908 against 1758.
constexpr size_t kPackAutoBytes = 48u << 20;
bool want_pack(const soma_ctx* c)
{
    if (c->n_types != 2 || c->count_bits == 32) return false;
    return c->count_bits == 16 || 16 * (size_t)c->cells > kPackAutoBytes;
}

// toff follows the grid format: call after c->pack changed.  Synchronises (host vector goes out of scope).
int upload_toff(soma_ctx* c)
{
    std::vector<uint32_t> t(c->types_host.size());
    for (size_t i = 0; i < t.size(); ++i) t[i] = c->types_host[i] * (c->pack ? 1u : (uint32_t)c->cells);
    CU(cudaMemcpyAsync(c->toff, t.data(), sizeof(uint32_t) * t.size(), cudaMemcpyHostToDevice, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return SOMA_OK;
}

size_t counts_bytes(const soma_ctx* c)
{
    return sizeof(uint32_t) * c->cells * (c->pack ? 1 : (size_t)c->n_types);
}

// check_domain: also count the beads whose coordinates lie outside the supported domain (stage 1 of new
// positions); the per-sweep histograms of SOMA_OPT_DENSITY = 1 do not -- moves cannot leave the domain
int launch_histogram(soma_ctx* c, bool check_domain_too)
{
    CU(cudaMemsetAsync(c->counts, 0, counts_bytes(c), c->stream));
    if (c->sharded) CU(cudaMemsetAsync(c->exchange, 0, counts_bytes(c), c->stream));   // counts = 0 + sum of the ranks' histograms
    if (c->sharded) c->counts_pending = true;
    const soma::GridP g = c->gridp();
    for (const Spec& s : c->specs) {
        if (s.n_beads == 0) continue;
        const int threads = 256;
        uint64_t blocks = (s.n_beads + threads - 1) / threads;
        const uint64_t cap = (uint64_t)c->n_sm * 16;
        if (blocks > cap) blocks = cap;
        Timed t(c, SOMA_K_DENSITY, 1);
        auto kernel = c->pack ? soma::histogram_kernel<true> : soma::histogram_kernel<false>;
        kernel<<<(unsigned)blocks, threads, 0, c->stream>>>(
            g, c->x + s.off, c->y + s.off, c->z + s.off, c->toff + s.toff_off, s.N, (uint32_t)s.n_beads, count_target(c),
            check_domain_too ? c->n_outside : nullptr);
        CU(cudaGetLastError());
    }
    return SOMA_OK;
}

// a4.  A shard folds the exchange array (summed over the ranks by now) into its copy of the whole system's
// occupation numbers on the way.
//   fold: 0 no exchange array, 1 fold this rank's (already summed) exchange array, 2 reduce the peers' arrays
int launch_fields(soma_ctx* c, int fold = 0)
{
    const soma::FieldP F = c->fieldp();
    const int threads = 256;
    const unsigned blocks = (unsigned)((c->cells + threads - 1) / threads);
    Timed t(c, SOMA_K_FIELD, 1);
    const bool pdl = c->pdl != 0;
    // One cell per thread: with programmatic dependent launch the many small blocks slip in behind the
    // draining move blocks.
    const unsigned long long n = c->n_beads_global;        // the beads counts holds (the packed format's overflow check)
    const size_t stride = (size_t)c->cells * c->n_types;   // words per exchange buffer
    uint32_t* ex = fold == 1 ? c->exchange : fold == 2 ? c->exchange_base + (size_t)(1 - c->peer_parity) * stride : nullptr;
    const uint32_t* const* peers = fold == 2 ? c->peer_table : nullptr;
    const uint32_t n_peers = (uint32_t)c->n_peers;
    const size_t peer_off = (size_t)c->peer_parity * stride;
    if (c->pack) {
        CU(launch_pdl(pdl, soma::field_kernel<2, true>, blocks, threads, 0, c->stream, F, c->counts, c->omega, c->ext, c->forbidden, c->ticket_sum, c->overflow_dev, n, ex, peers, n_peers, peer_off));
        return SOMA_OK;
    }
    switch (c->n_types) {
        case 1: CU(launch_pdl(pdl, soma::field_kernel<1, false>, blocks, threads, 0, c->stream, F, c->counts, c->omega, c->ext, c->forbidden, c->ticket_sum, c->overflow_dev, n, ex, peers, n_peers, peer_off)); break;
        case 2: CU(launch_pdl(pdl, soma::field_kernel<2, false>, blocks, threads, 0, c->stream, F, c->counts, c->omega, c->ext, c->forbidden, c->ticket_sum, c->overflow_dev, n, ex, peers, n_peers, peer_off)); break;
        default: CU(launch_pdl(pdl, soma::field_kernel<0, false>, blocks, threads, 0, c->stream, F, c->counts, c->omega, c->ext, c->forbidden, c->ticket_sum, c->overflow_dev, n, ex, peers, n_peers, peer_off)); break;
    }
    return SOMA_OK;
}

// omega after a parameter change (a shard holds the whole system's occupation numbers too).  Between a histogram
// of a shard (soma_init_shard, soma_set_positions, a change of SOMA_OPT_COUNT_BITS) and the soma_shard_fields(ctx, 0)
// that follows it, counts is all zero: omega of that would be meaningless, and the packed format's check (halves
// against the number of beads) would raise the sticky overflow flag.  Nothing to do then: that soma_shard_fields
// computes omega with the parameters as they are by then.
int refresh_fields(soma_ctx* c)
{
    if (c->sharded && c->counts_pending) return SOMA_OK;
    return launch_fields(c);
}

// After new positions came in (soma_init, soma_set_positions): did the histogram see a coordinate outside
// the supported domain |x_a n_a / L_a| < 2^22, or a NaN?  Synchronises.
int check_domain(soma_ctx* c, const char* who)
{
    uint32_t bad = 0;
    CU(cudaMemcpyAsync(&bad, c->n_outside, sizeof(uint32_t), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    if (bad == 0) return SOMA_OK;
    return fail(SOMA_EDOMAIN, "%s: %u beads have a coordinate that is not finite or lies outside the supported "
                "domain |x n / L| < 2^22 per axis", who, bad);
}

// The sticky flag of the packed occupation numbers (soma::field_kernel): valid after a synchronisation.
int check_overflow(soma_ctx* c, const char* who)
{
    if (!*(volatile uint32_t*)c->overflow_host) return SOMA_OK;
    return fail(SOMA_EOVERFLOW, "%s: a cell holds more than 65535 beads of one type, which the packed 16-bit "
                "occupation numbers cannot count; set SOMA_OPT_COUNT_BITS to 32 and restart from a configuration "
                "saved before", who);
}

int stage1_once(soma_ctx* c)
{
    CU(cudaMemsetAsync(c->n_outside, 0, sizeof(uint32_t), c->stream));
    int rc = launch_histogram(c, true);
    if (rc) return rc;
    if (c->sharded) return SOMA_OK;   // omega needs every rank's contribution: soma_shard_fields
    return launch_fields(c);
}

// Stage 1 on new positions (soma_init, soma_set_positions): occupation numbers, fields, and the checks of
// the coordinate domain and of the packed counters.  Synchronises.  With SOMA_OPT_COUNT_BITS = 0 (auto) a
// configuration too dense for 16 + 16 bits switches the context to 32-bit counters.
int stage1(soma_ctx* c, const char* who)
{
    int rc = stage1_once(c);
    if (rc) return rc;
    rc = check_domain(c, who);
    if (rc) return rc;
    if (c->pack && *(volatile uint32_t*)c->overflow_host) {
        if (c->count_bits == 16) return check_overflow(c, who);
        *(volatile uint32_t*)c->overflow_host = 0u;
        c->pack = false;
        rc = upload_toff(c);
        if (rc) return rc;
        rc = stage1_once(c);
        if (rc) return rc;
        CU(cudaStreamSynchronize(c->stream));
    }
    return SOMA_OK;
}

// ---- layout: Hilbert order of the chains, caller order <-> device order ---------------------------
int ensure_stage(soma_ctx* c)
{
    if (!c->stage) CU(cudaMalloc(&c->stage, sizeof(float) * 3 * c->n_beads));
    return SOMA_OK;
}

// Put the chains of every architecture in Hilbert order of their centres of mass.
int resort(soma_ctx* c)
{
    c->sweeps_since_sort = 0;
    if (c->layout == 0) return SOMA_OK;
    int max_n = std::max(c->grid[0], std::max(c->grid[1], c->grid[2]));
    uint32_t bits = 1;
    while (bits < 10 && (1 << bits) < max_n) ++bits;
    // Units of the 2^bits Hilbert cube the box spans per axis: the same length per unit along x and y (the
    // longest axis fills the cube) and twice that along z, the direction in which the cells of omega and
    // counts are contiguous in memory (a 32-byte sector is 8 cells along z).  Measured at C4 (box 64 x 64 x
    // 16): 2018 us per step with every axis scaled to the full cube, 1924 isotropic, 1900 with this.
    const float l_max = std::max(c->box[0], std::max(c->box[1], c->box[2]));
    const float side[3] = {(float)(1u << bits) * c->box[0] / l_max, (float)(1u << bits) * c->box[1] / l_max,
                           (float)(1u << bits) * c->box[2] / l_max * 0.5f};
    for (const Spec& s : c->specs) {
        if (s.n_chains < 2) continue;
        const uint32_t n = (uint32_t)s.n_chains;
        Timed t(c, SOMA_K_LAYOUT, 5);
        soma::chain_key_kernel<<<(n + 127) / 128, 128, 0, c->stream>>>(
            c->x + s.off, c->y + s.off, c->z + s.off, n, s.N, (float)(1.0 / (double)c->box[0]),
            (float)(1.0 / (double)c->box[1]), (float)(1.0 / (double)c->box[2]), bits, side[0], side[1], side[2],
            c->sort_keys[0], c->sort_vals[0]);
        size_t tmp = c->cub_tmp_bytes;
        CU(cub::DeviceRadixSort::SortPairs(c->cub_tmp, tmp, c->sort_keys[0], c->sort_keys[1], c->sort_vals[0],
                                           c->sort_vals[1], (int)n, 0, (int)(3 * bits), c->stream));
        const uint32_t* order = c->sort_vals[1];          // order[new slot] = old slot
        const unsigned blocks = (unsigned)((s.n_beads + 255) / 256);
        float** arr[3] = {&c->x, &c->y, &c->z};
        for (int a = 0; a < 3; ++a) {
            // gather this architecture's segment into the scratch array, then copy it back in place
            soma::permute_chains_kernel<<<blocks, 256, 0, c->stream>>>(c->scratch + s.off, *arr[a] + s.off, order, s.N, s.n_beads);
            CU(cudaMemcpyAsync(*arr[a] + s.off, c->scratch + s.off, sizeof(float) * s.n_beads, cudaMemcpyDeviceToDevice, c->stream));
        }
        soma::permute_ids_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(c->orig_tmp, c->orig + s.chain_off, order, n);
        CU(cudaMemcpyAsync(c->orig + s.chain_off, c->orig_tmp, sizeof(uint32_t) * n, cudaMemcpyDeviceToDevice, c->stream));
        CU(cudaGetLastError());
    }
    return SOMA_OK;
}

// caller's SoA x | y | z  <->  device layout, through orig[]
int copy_soa(soma_ctx* c, float* dst_user, const float* src_user, bool to_user, bool user_is_device)
{
    float* user = to_user ? dst_user : const_cast<float*>(src_user);
    float* dev_user = user;
    if (!user_is_device) {
        int rc = ensure_stage(c);
        if (rc) return rc;
        dev_user = c->stage;
        if (!to_user)
            CU(cudaMemcpyAsync(c->stage, src_user, sizeof(float) * 3 * c->n_beads, cudaMemcpyHostToDevice, c->stream));
    }
    for (const Spec& s : c->specs) {
        if (s.n_beads == 0) continue;
        const unsigned blocks = (unsigned)((s.n_beads + 255) / 256);
        Timed t(c, SOMA_K_LAYOUT, 1);
        if (to_user)
            soma::reorder_kernel<true><<<blocks, 256, 0, c->stream>>>(dev_user, c->n_beads, c->x + s.off, c->y + s.off,
                                                                     c->z + s.off, c->orig + s.chain_off, s.N, s.n_beads, s.local0);
        else
            soma::reorder_kernel<false><<<blocks, 256, 0, c->stream>>>(dev_user, c->n_beads, c->x + s.off, c->y + s.off,
                                                                      c->z + s.off, c->orig + s.chain_off, s.N, s.n_beads, s.local0);
    }
    CU(cudaGetLastError());
    if (!user_is_device && to_user)
        CU(cudaMemcpyAsync(dst_user, c->stage, sizeof(float) * 3 * c->n_beads, cudaMemcpyDeviceToHost, c->stream));
    return SOMA_OK;
}

}  // namespace

// =================================================================================================
// C ABI
// =================================================================================================
extern "C" {

const char* soma_last_error(void) { return g_err.c_str(); }
const char* soma_version(void) { return "soma-b200 0.2 (sm_100a)"; }

int soma_architecture_words(const soma_chain_spec* spec, uint32_t* words_out, uint64_t capacity, uint64_t* n_words,
                            uint32_t* n_sets)
{
    if (!spec || !n_words) return fail(SOMA_EINVAL, "soma_architecture_words: NULL argument");
    if (spec->n_beads < 1 || spec->n_bonds < 1)
        return fail(SOMA_EINVAL, "soma_architecture_words: need n_beads >= 1 and a bond list (a linear chain keeps no array)");
    std::vector<uint32_t> words, set_off;
    int rc = build_architecture(*spec, 0, words, set_off);
    if (rc) return rc;
    *n_words = words.size();
    if (n_sets) *n_sets = (uint32_t)(set_off.size() - 1);
    if (words_out) {
        if (capacity < words.size()) return fail(SOMA_EINVAL, "soma_architecture_words: %zu words needed, room for %llu", words.size(), (unsigned long long)capacity);
        std::memcpy(words_out, words.data(), sizeof(uint32_t) * words.size());
    }
    return SOMA_OK;
}

void soma_destroy(soma_ctx* c)
{
    if (!c) return;
    DeviceGuard on_device(c->device);
    cudaStreamSynchronize(c->stream);
    for (auto& e : c->ev) cudaEventDestroy(e);
    cudaFree(c->x); cudaFree(c->y); cudaFree(c->z);
    for (void* m : c->peer_opened) cudaIpcCloseMemHandle(m);
    cudaFree(c->peer_table);
    cudaFree(c->exchange_base);
    cudaFree(c->n_outside);
    cudaFree(c->ticket_sum);
    cudaFree(c->grid_stage);
    if (c->overflow_host) cudaFreeHost(c->overflow_host);
    cudaFree(c->counts); cudaFree(c->omega); cudaFree(c->toff); cudaFree(c->decisions);
    cudaFree(c->ext); cudaFree(c->forbidden); cudaFree(c->arch);
    cudaFree(c->acc_slots);
    cudaFree(c->orig); cudaFree(c->orig_tmp); cudaFree(c->scratch); cudaFree(c->stage);
    cudaFree(c->sort_keys[0]); cudaFree(c->sort_keys[1]); cudaFree(c->sort_vals[0]); cudaFree(c->sort_vals[1]);
    cudaFree(c->cub_tmp);
    if (c->acc_host) cudaFreeHost(c->acc_host);
    delete c;
}

static int init_impl(soma_ctx** out, const soma_chain_spec* chains, int n_specs, int N_ref, int n_types,
                     const float* box, const int* grid, float chiN, float kappaN, float A, uint64_t seed,
                     const float* host_xyz0, void* cuda_stream, const uint64_t* spec_first_bead,
                     uint64_t global_n_beads)
{
    if (!out) return fail(SOMA_EINVAL, "soma_init: out is NULL");
    *out = nullptr;
    if (!chains || n_specs < 1) return fail(SOMA_EINVAL, "soma_init: need at least one chain spec");
    if (N_ref < 1) return fail(SOMA_EINVAL, "soma_init: N_ref must be >= 1");
    if (n_types < 1 || n_types > SOMA_MAX_TYPES)
        return fail(SOMA_EINVAL, "soma_init: n_types must be in 1..%d", SOMA_MAX_TYPES);
    if (!box || !grid) return fail(SOMA_EINVAL, "soma_init: box/grid is NULL");
    double min_box = 1e300;
    uint64_t cells = 1;
    for (int a = 0; a < 3; ++a) {
        if (!(box[a] > 0.0f) || !std::isfinite(box[a])) return fail(SOMA_EINVAL, "soma_init: box[%d] must be > 0", a);
        if (grid[a] < 1 || grid[a] > (1 << 22)) return fail(SOMA_EINVAL, "soma_init: grid[%d] must be in 1..2^22", a);
        min_box = box[a] < min_box ? box[a] : min_box;
        cells *= (uint64_t)grid[a];
        if (cells >= (1ull << 31)) return fail(SOMA_EINVAL, "soma_init: too many grid cells (>= 2^31)");
    }
    if (cells * (uint64_t)n_types >= (1ull << 32))
        return fail(SOMA_EINVAL, "soma_init: n_types * cells must be < 2^32");
    if (!(A > 0.0f) || !((double)A <= 0.5 * min_box))
        return fail(SOMA_EINVAL, "soma_init: need 0 < A <= min(box)/2");
    if (!std::isfinite(chiN) || !std::isfinite(kappaN)) return fail(SOMA_EINVAL, "soma_init: chiN/kappaN not finite");

    soma_ctx* c = new (std::nothrow) soma_ctx;
    if (!c) return fail(SOMA_ENOMEM, "soma_init: out of host memory");
    c->n_types = n_types;
    c->N_ref = N_ref;
    c->kappaN = kappaN;
    c->A = A;
    c->seed = seed;
    c->cells = cells;
    c->stream = (cudaStream_t)cuda_stream;
    for (int a = 0; a < 3; ++a) { c->box[a] = box[a]; c->grid[a] = grid[a]; }
    for (int i = 0; i < n_types; ++i)
        for (int k = 0; k < n_types; ++k) c->chiN[i][k] = i == k ? 0.0f : chiN;

    std::vector<uint32_t> toff_host, arch_host;
    uint64_t gid = 0, off = 0;
    for (int a = 0; a < n_specs; ++a) {
        Spec s;
        s.n_chains = chains[a].n_chains;
        s.N = chains[a].n_beads;
        if (s.N < 1 || (s.n_chains > 0 && !chains[a].types)) {
            delete c;
            return fail(SOMA_EINVAL, "soma_init: spec %d: n_beads must be >= 1 and types non-NULL", a);
        }
        s.n_beads = s.n_chains * s.N;
        s.gid0 = spec_first_bead ? spec_first_bead[a] : gid;
        s.local0 = gid;
        if (spec_first_bead && (s.gid0 + s.n_beads > global_n_beads || global_n_beads >= (1ull << 32))) {
            delete c;
            return fail(SOMA_EINVAL, "soma_init_shard: spec %d does not fit into the global system (first bead %llu, "
                        "%llu beads, %llu beads in all, which must be < 2^32)", a, (unsigned long long)s.gid0,
                        (unsigned long long)s.n_beads, (unsigned long long)global_n_beads);
        }
        s.off = off;
        s.toff_off = (uint32_t)toff_host.size();
        s.n_bonds = chains[a].n_bonds;
        s.general = s.n_bonds > 0;
        if (s.general) {
            s.arch_off = arch_host.size();
            int rc_arch = build_architecture(chains[a], a, arch_host, s.set_off);
            if (rc_arch) { delete c; return rc_arch; }
            s.n_arch_words = (uint32_t)(arch_host.size() - s.arch_off);
        }
        s.fused_ok = !s.general && s.N >= 4 && s.N <= 128 && (s.N % 4) == 0;
        s.any_n = s.fused_ok && (128 % s.N) != 0;
        if (s.any_n) {
            s.log2N = 128 / s.N;                                   // chains per tile
            s.n_tiles = (uint32_t)(s.n_chains / s.log2N);
        } else if (s.fused_ok) {
            while ((1u << s.log2N) < s.N) ++s.log2N;
            s.n_tiles = (uint32_t)(s.n_chains * s.N / soma::kTile);
        }
        s.chain_off = c->n_chains_total;
        c->n_chains_total += s.n_chains;
        c->max_chains = std::max<uint64_t>(c->max_chains, s.n_chains);
        if (s.n_chains >= (1ull << 32)) {
            delete c;
            return fail(SOMA_EINVAL, "soma_init: spec %d has 2^32 or more chains", a);
        }
        for (uint32_t j = 0; j < s.N; ++j) {
            const uint8_t t = s.n_chains ? chains[a].types[j] : 0;
            if (t >= n_types) {
                delete c;
                return fail(SOMA_EINVAL, "soma_init: spec %d monomer %u has type %u >= n_types", a, j, (unsigned)t);
            }
            toff_host.push_back((uint32_t)t);
        }
        while (toff_host.size() % 4) toff_host.push_back(0);  // uint4 loads of the fused kernel
        gid += s.n_beads;
        off += (s.n_beads + 127) / 128 * 128;
        if (gid >= (1ull << 32)) {
            delete c;
            return fail(SOMA_EINVAL, "soma_init: total beads must be < 2^32");
        }
        c->specs.push_back(s);
    }
    c->n_beads = gid;
    c->sharded = spec_first_bead != nullptr;
    c->n_beads_global = c->sharded ? global_n_beads : gid;
    c->n_pad = off + 128;
    if (c->n_beads == 0) {
        delete c;
        return fail(SOMA_EINVAL, "soma_init: the system has no beads");
    }

    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev < 1) {
        cudaGetLastError();
        delete c;
        return fail(SOMA_ENODEVICE, "soma_init: no CUDA device (this library has no CPU path)");
    }
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { delete c; return fail(SOMA_ECUDA, "soma_init: cudaGetDevice failed"); }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) { delete c; return fail(SOMA_ECUDA, "soma_init: cudaGetDeviceProperties failed"); }
    if (prop.major != 10) {
        delete c;
        return fail(SOMA_ENODEVICE, "soma_init: kernels are built for sm_100a only, device is sm_%d%d", prop.major, prop.minor);
    }
    c->device = dev;
    c->n_sm = prop.multiProcessorCount;


#define CUI(call)                                                                      \
    do {                                                                               \
        cudaError_t e_ = (call);                                                       \
        if (e_ != cudaSuccess) {                                                       \
            int rc_ = fail(e_ == cudaErrorMemoryAllocation ? SOMA_ENOMEM : SOMA_ECUDA, \
                           "%s: %s", #call, cudaGetErrorString(e_));                   \
            cudaGetLastError();                                                        \
            soma_destroy(c);                                                           \
            return rc_;                                                                \
        }                                                                              \
    } while (0)

    CUI(cudaMalloc(&c->orig, sizeof(uint32_t) * c->n_chains_total));
    CUI(cudaMalloc(&c->orig_tmp, sizeof(uint32_t) * c->max_chains));
    CUI(cudaMalloc(&c->scratch, sizeof(float) * c->n_pad));
    for (int i = 0; i < 2; ++i) {
        CUI(cudaMalloc(&c->sort_keys[i], sizeof(uint32_t) * c->max_chains));
        CUI(cudaMalloc(&c->sort_vals[i], sizeof(uint32_t) * c->max_chains));
    }
    CUI(cub::DeviceRadixSort::SortPairs(nullptr, c->cub_tmp_bytes, c->sort_keys[0], c->sort_keys[1], c->sort_vals[0],
                                        c->sort_vals[1], (int)c->max_chains, 0, 30, c->stream));
    CUI(cudaMalloc(&c->cub_tmp, c->cub_tmp_bytes + 16));
    for (const Spec& s : c->specs)
        if (s.n_chains)
            soma::iota_kernel<<<(unsigned)((s.n_chains + 255) / 256), 256, 0, c->stream>>>(c->orig + s.chain_off, (uint32_t)s.n_chains);
    CUI(cudaMalloc(&c->x, sizeof(float) * c->n_pad));
    CUI(cudaMalloc(&c->y, sizeof(float) * c->n_pad));
    CUI(cudaMalloc(&c->z, sizeof(float) * c->n_pad));
    CUI(cudaMalloc(&c->counts, sizeof(uint32_t) * cells * n_types));
    if (c->sharded) {
        CUI(cudaMalloc(&c->exchange_base, 2 * sizeof(uint32_t) * cells * n_types));
        CUI(cudaMemsetAsync(c->exchange_base, 0, 2 * sizeof(uint32_t) * cells * n_types, c->stream));
        c->exchange = c->exchange_base;
    }
    CUI(cudaMalloc(&c->omega, sizeof(float) * cells * n_types));
    CUI(cudaMalloc(&c->toff, sizeof(uint32_t) * toff_host.size()));
    if (!arch_host.empty()) {
        CUI(cudaMalloc(&c->arch, sizeof(uint32_t) * arch_host.size()));
        CUI(cudaMemcpyAsync(c->arch, arch_host.data(), sizeof(uint32_t) * arch_host.size(), cudaMemcpyHostToDevice, c->stream));
    }
    CUI(cudaMalloc(&c->decisions, sizeof(uint32_t) * ((c->n_beads_global + 31) / 32 + 8)));
    CUI(cudaMalloc(&c->acc_slots, sizeof(unsigned long long) * soma::kAccSlots));
    CUI(cudaMalloc(&c->n_outside, sizeof(uint32_t)));
    CUI(cudaMalloc(&c->ticket_sum, sizeof(unsigned long long)));
    CUI(cudaMemsetAsync(c->ticket_sum, 0, sizeof(unsigned long long), c->stream));
    CUI(cudaHostAlloc(&c->overflow_host, sizeof(uint32_t), cudaHostAllocMapped));
    *c->overflow_host = 0u;
    CUI(cudaHostGetDevicePointer((void**)&c->overflow_dev, c->overflow_host, 0));
    c->pack = want_pack(c);
    CUI(cudaMemsetAsync(c->n_outside, 0, sizeof(uint32_t), c->stream));
    CUI(cudaMallocHost(&c->acc_host, sizeof(unsigned long long) * soma::kAccSlots));
    CUI(cudaMemsetAsync(c->x, 0, sizeof(float) * c->n_pad, c->stream));
    CUI(cudaMemsetAsync(c->y, 0, sizeof(float) * c->n_pad, c->stream));
    CUI(cudaMemsetAsync(c->z, 0, sizeof(float) * c->n_pad, c->stream));
    CUI(cudaMemsetAsync(c->decisions, 0, sizeof(uint32_t) * ((c->n_beads_global + 31) / 32 + 8), c->stream));
    CUI(cudaMemsetAsync(c->acc_slots, 0, sizeof(unsigned long long) * soma::kAccSlots, c->stream));
    c->types_host = toff_host;
    if (upload_toff(c) != SOMA_OK) { soma_destroy(c); return SOMA_ECUDA; }

    int rc = SOMA_OK;
    if (host_xyz0) {
        rc = copy_soa(c, nullptr, host_xyz0, false, false);
    } else {
        const double sigma = N_ref > 1 ? 1.0 / std::sqrt(3.0 * ((double)N_ref - 1.0)) : 0.0;
        for (const Spec& s : c->specs) {
            if (s.n_chains == 0) continue;
            const int threads = 128;
            const unsigned blocks = (unsigned)((s.n_chains + threads - 1) / threads);
            c->launches += 1;
            soma::init_walk_kernel<<<blocks, threads, 0, c->stream>>>(
                c->x + s.off, c->y + s.off, c->z + s.off, s.n_chains, s.N, (uint32_t)s.gid0, (uint32_t)seed,
                (uint32_t)(seed >> 32), (double)box[0], (double)box[1], (double)box[2], sigma);
        }
        if (cudaGetLastError() != cudaSuccess) rc = fail(SOMA_ECUDA, "soma_init: init_walk_kernel launch failed");
    }
    if (rc == SOMA_OK) rc = resort(c);
    if (rc == SOMA_OK) rc = stage1(c, "soma_init");
    if (rc == SOMA_OK && cudaStreamSynchronize(c->stream) != cudaSuccess)
        rc = fail(SOMA_ECUDA, "soma_init: %s", cudaGetErrorString(cudaGetLastError()));
    if (rc != SOMA_OK) {
        std::string keep = g_err;
        soma_destroy(c);
        g_err = keep;
        return rc;
    }
    *out = c;
    return SOMA_OK;
#undef CUI
}

int soma_init(soma_ctx** out, const soma_chain_spec* chains, int n_specs, int N_ref, int n_types,
              const float* box, const int* grid, float chiN, float kappaN, float A, uint64_t seed,
              const float* host_xyz0, void* cuda_stream)
{
    return init_impl(out, chains, n_specs, N_ref, n_types, box, grid, chiN, kappaN, A, seed, host_xyz0, cuda_stream,
                     nullptr, 0);
}

int soma_init_shard(soma_ctx** out, const soma_chain_spec* chains, int n_specs, int N_ref, int n_types,
                    const float* box, const int* grid, float chiN, float kappaN, float A, uint64_t seed,
                    const float* host_xyz0, void* cuda_stream, const uint64_t* spec_first_bead,
                    uint64_t global_n_beads)
{
    if (!spec_first_bead) return fail(SOMA_EINVAL, "soma_init_shard: spec_first_bead is NULL");
    return init_impl(out, chains, n_specs, N_ref, n_types, box, grid, chiN, kappaN, A, seed, host_xyz0, cuda_stream,
                     spec_first_bead, global_n_beads);
}

// the moves of one sweep: a1, a2 (or a5) [+ a3]
static int sweep_moves(soma_ctx* c)
{
    if (c->record)
        CU(cudaMemsetAsync(c->decisions, 0, sizeof(uint32_t) * ((c->n_beads_global + 31) / 32), c->stream));
    if (c->layout && c->sort_interval > 0 && c->sweeps_since_sort >= (uint64_t)c->sort_interval) {
        int rs = resort(c);                            // storage order only: no result depends on it
        if (rs) return rs;
    }
    c->sweeps_since_sort += 1;
    const soma::MoveP P = c->movep(c->sweep);
    int rc = launch_moves(c, P);                       // a1, a2 (or a5) [+ a3 incremental]
    if (rc) return rc;
    if (c->density_mode == 1) {
        rc = launch_histogram(c, false);               // a3 from scratch
        if (rc) return rc;
    }
    return SOMA_OK;
}

static int check_step(soma_ctx* c, const char* who)
{
    if (c->move == 2 && !(c->smc_step > 0.0f))
        return fail(SOMA_ESTATE, "%s: Smart-MC selected but SOMA_OPT_SMC_STEP not set", who);
    if (c->scheme == 1 || c->set_order == 1)
        for (const Spec& s : c->specs)
            if (s.general)
                return fail(SOMA_ESTATE, "%s: architectures given by a bond list support SOMA_OPT_SCHEME 0 and SOMA_OPT_SET_ORDER 0 only", who);
    if (c->sharded) {
        // a part of a larger system is parity-checked for linear chains in the set scheme only
        if (c->scheme == 1)
            return fail(SOMA_ESTATE, "%s: a shard supports SOMA_OPT_SCHEME 0 only", who);
        for (const Spec& s : c->specs)
            if (s.general)
                return fail(SOMA_ESTATE, "%s: a shard supports linear chains only (no bond-list architectures)", who);
    }
    return SOMA_OK;
}

int soma_step(soma_ctx* c, int n_sweeps)
{
    if (!c) return fail(SOMA_EINVAL, "soma_step: ctx is NULL");
    DeviceGuard on_device(c->device);
    if (n_sweeps < 0) return fail(SOMA_EINVAL, "soma_step: n_sweeps must be >= 0");
    if (c->sharded) return fail(SOMA_ESTATE, "soma_step: this context is a shard: use soma_shard_moves / soma_shard_fields");
    int rc = check_step(c, "soma_step");
    if (rc) return rc;
    rc = check_overflow(c, "soma_step");                   // of the sweeps that have completed so far
    if (rc) return rc;
    for (int i = 0; i < n_sweeps; ++i) {
        rc = sweep_moves(c);
        if (rc) return rc;
        if (c->field_interval <= 1 || (c->sweep + 1) % (uint64_t)c->field_interval == 0) {
            rc = launch_fields(c);                         // a4
            if (rc) return rc;
        }
        c->sweep += 1;
        c->attempted += c->n_beads;
        c->decisions_valid = c->record != 0;
    }
    return SOMA_OK;
}

int soma_shard_moves(soma_ctx* c)
{
    if (!c) return fail(SOMA_EINVAL, "soma_shard_moves: ctx is NULL");
    DeviceGuard on_device(c->device);
    if (!c->sharded) return fail(SOMA_ESTATE, "soma_shard_moves: the context was not created by soma_init_shard");
    int rc = check_step(c, "soma_shard_moves");
    if (rc) return rc;
    rc = sweep_moves(c);
    if (rc) return rc;
    c->attempted += c->n_beads;
    c->decisions_valid = c->record != 0;
    return SOMA_OK;
}

int soma_shard_exchange(soma_ctx* c, void** dev_words, uint64_t* n_words)
{
    if (!c || !dev_words || !n_words) return fail(SOMA_EINVAL, "soma_shard_exchange: NULL argument");
    if (!c->sharded) return fail(SOMA_ESTATE, "soma_shard_exchange: the context was not created by soma_init_shard");
    *dev_words = c->exchange;
    *n_words = counts_bytes(c) / sizeof(uint32_t);
    return SOMA_OK;
}

int soma_shard_exchange_copy(soma_ctx* c, uint32_t* host_words, int to_host)
{
    if (!c || !host_words) return fail(SOMA_EINVAL, "soma_shard_exchange_copy: NULL argument");
    DeviceGuard on_device(c->device);
    if (!c->sharded) return fail(SOMA_ESTATE, "soma_shard_exchange_copy: the context was not created by soma_init_shard");
    if (to_host) CU(cudaMemcpyAsync(host_words, c->exchange, counts_bytes(c), cudaMemcpyDeviceToHost, c->stream));
    else CU(cudaMemcpyAsync(c->exchange, host_words, counts_bytes(c), cudaMemcpyHostToDevice, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return SOMA_OK;
}

int soma_shard_peer_handle(soma_ctx* c, void* handle64)
{
    if (!c || !handle64) return fail(SOMA_EINVAL, "soma_shard_peer_handle: NULL argument");
    DeviceGuard on_device(c->device);
    if (!c->sharded) return fail(SOMA_ESTATE, "soma_shard_peer_handle: the context was not created by soma_init_shard");
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "CUDA IPC handles are 64 bytes");
    cudaIpcMemHandle_t h;
    CU(cudaIpcGetMemHandle(&h, c->exchange_base));
    std::memcpy(handle64, &h, sizeof h);
    return SOMA_OK;
}

int soma_shard_set_peers(soma_ctx* c, int n_ranks, int my_rank, void* const* peer_dev, const void* handles)
{
    if (!c) return fail(SOMA_EINVAL, "soma_shard_set_peers: ctx is NULL");
    DeviceGuard on_device(c->device);
    if (!c->sharded) return fail(SOMA_ESTATE, "soma_shard_set_peers: the context was not created by soma_init_shard");
    if (n_ranks < 1 || my_rank < 0 || my_rank >= n_ranks || (!peer_dev && !handles))
        return fail(SOMA_EINVAL, "soma_shard_set_peers: need 0 <= my_rank < n_ranks and the peers' addresses or handles");
    if (c->n_peers) return fail(SOMA_ESTATE, "soma_shard_set_peers: the peers of this context are already set");
    if (c->sweep != 0) return fail(SOMA_ESTATE, "soma_shard_set_peers: call it before the first sweep");
    std::vector<const uint32_t*> table(n_ranks);
    // on any failure below the context is left as it was: mappings opened by this call are closed again and the
    // table is freed, so that the call can be repeated
    auto undo = [c](int code) {
        for (void* m : c->peer_opened) cudaIpcCloseMemHandle(m);
        c->peer_opened.clear();
        if (c->peer_table) cudaFree(c->peer_table);
        c->peer_table = nullptr;
        cudaGetLastError();
        return code;
    };
    for (int r = 0; r < n_ranks; ++r) {
        if (r == my_rank) { table[r] = c->exchange_base; continue; }
        if (peer_dev && peer_dev[r]) { table[r] = (const uint32_t*)peer_dev[r]; continue; }
        if (!handles) return undo(fail(SOMA_EINVAL, "soma_shard_set_peers: no address and no handle for rank %d", r));
        cudaIpcMemHandle_t h;
        std::memcpy(&h, (const char*)handles + 64 * (size_t)r, sizeof h);
        void* mapped = nullptr;
        cudaError_t e = cudaIpcOpenMemHandle(&mapped, h, cudaIpcMemLazyEnablePeerAccess);
        if (e != cudaSuccess)
            return undo(fail(SOMA_ECUDA, "soma_shard_set_peers: cudaIpcOpenMemHandle for rank %d: %s", r, cudaGetErrorString(e)));
        c->peer_opened.push_back(mapped);
        table[r] = (const uint32_t*)mapped;
    }
    cudaError_t e = cudaMalloc(&c->peer_table, sizeof(uint32_t*) * n_ranks);
    if (e == cudaSuccess)
        e = cudaMemcpyAsync(c->peer_table, table.data(), sizeof(uint32_t*) * n_ranks, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess)
        return undo(fail(e == cudaErrorMemoryAllocation ? SOMA_ENOMEM : SOMA_ECUDA, "soma_shard_set_peers: table of the peers' "
                         "addresses: %s", cudaGetErrorString(e)));
    c->n_peers = n_ranks;
    c->my_rank = my_rank;
    return SOMA_OK;
}

int soma_shard_fields(soma_ctx* c, int advance)
{
    if (!c) return fail(SOMA_EINVAL, "soma_shard_fields: ctx is NULL");
    DeviceGuard on_device(c->device);
    if (!c->sharded) return fail(SOMA_ESTATE, "soma_shard_fields: the context was not created by soma_init_shard");
    if (c->n_peers) {
        // the field kernel reduces the ranks' exchange arrays itself (peer memory), folds the sum into the whole
        // system's numbers and clears this rank's other buffer, into which the next sweep counts
        if (c->field_interval > 1)
            return fail(SOMA_ESTATE, "soma_shard_fields: with peers set, SOMA_OPT_FIELD_INTERVAL must be 1");
        int rc = launch_fields(c, 2);
        if (rc) return rc;
        c->counts_pending = false;
        c->peer_parity ^= 1;
        c->exchange = c->exchange_base + (size_t)c->peer_parity * c->cells * c->n_types;
        if (advance) c->sweep += 1;
        return SOMA_OK;
    }
    if (!advance || c->field_interval <= 1 || (c->sweep + 1) % (uint64_t)c->field_interval == 0) {
        int rc = launch_fields(c, 1);                      // a4 from the occupation numbers of the whole system
        if (rc) return rc;
    } else {                                               // the counts stay current; omega is not due
        const uint64_t n = counts_bytes(c) / sizeof(uint32_t);
        c->launches += 1;
        soma::fold_exchange_kernel<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(c->counts, c->exchange, n);
        CU(cudaGetLastError());
    }
    c->counts_pending = false;
    if (advance) c->sweep += 1;
    return SOMA_OK;
}

int soma_fields(soma_ctx* c, float* omega, uint32_t* counts, int dst_is_device)
{
    if (!c) return fail(SOMA_EINVAL, "soma_fields: ctx is NULL");
    DeviceGuard on_device(c->device);
    if (!omega && !counts) return fail(SOMA_EINVAL, "soma_fields: both outputs NULL");
    // internal layout (records per cell, packed occupation numbers) -> the caller's [type][cell] arrays
    const size_t n = (size_t)c->cells * c->n_types;
    float* dev_omega = omega;
    uint32_t* dev_counts = counts;
    if (!dst_is_device) {
        if (!c->grid_stage) CU(cudaMalloc(&c->grid_stage, 2 * sizeof(float) * n));
        dev_omega = omega ? (float*)c->grid_stage : nullptr;
        dev_counts = counts ? (uint32_t*)c->grid_stage + n : nullptr;
    }
    const unsigned blocks = (unsigned)((n + 255) / 256);
    c->launches += 1;
    if (c->pack) soma::export_grid_kernel<true><<<blocks, 256, 0, c->stream>>>(c->omega, c->counts, (uint32_t)c->cells, (uint32_t)c->n_types, dev_omega, dev_counts);
    else soma::export_grid_kernel<false><<<blocks, 256, 0, c->stream>>>(c->omega, c->counts, (uint32_t)c->cells, (uint32_t)c->n_types, dev_omega, dev_counts);
    CU(cudaGetLastError());
    if (!dst_is_device) {
        if (omega) CU(cudaMemcpyAsync(omega, dev_omega, sizeof(float) * n, cudaMemcpyDeviceToHost, c->stream));
        if (counts) CU(cudaMemcpyAsync(counts, dev_counts, sizeof(uint32_t) * n, cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
        return check_overflow(c, "soma_fields");
    }
    return SOMA_OK;
}

int soma_positions(soma_ctx* c, float* xyz, int dst_is_device)
{
    if (!c || !xyz) return fail(SOMA_EINVAL, "soma_positions: NULL argument");
    DeviceGuard on_device(c->device);
    int rc = copy_soa(c, xyz, nullptr, true, dst_is_device != 0);
    if (rc) return rc;
    if (!dst_is_device) {
        CU(cudaStreamSynchronize(c->stream));
        return check_overflow(c, "soma_positions");
    }
    return SOMA_OK;
}

int soma_set_positions(soma_ctx* c, const float* xyz, int src_is_device)
{
    if (!c || !xyz) return fail(SOMA_EINVAL, "soma_set_positions: NULL argument");
    DeviceGuard on_device(c->device);
    int rc = copy_soa(c, nullptr, xyz, false, src_is_device != 0);
    if (rc) return rc;
    // The new positions keep the old storage order (usually they are a configuration this context
    // exported); if they are unrelated the order is stale, which only costs cache hits: bring the
    // next periodic re-sort forward to eight sweeps from now instead of sorting on every call.
    if (c->layout && c->sort_interval > 8)
        c->sweeps_since_sort = std::max<uint64_t>(c->sweeps_since_sort, (uint64_t)c->sort_interval - 8);
    if (c->pack != want_pack(c)) {   // auto: try the packed counters again if an earlier configuration was too dense
        c->pack = want_pack(c);
        rc = upload_toff(c);
        if (rc) return rc;
    }
    return stage1(c, "soma_set_positions");   // synchronises: the caller may reuse its buffer
}

int soma_set_chi(soma_ctx* c, int i, int j, float chiN_ij)
{
    if (!c) return fail(SOMA_EINVAL, "soma_set_chi: ctx is NULL");
    DeviceGuard on_device(c->device);
    if (i < 0 || j < 0 || i >= c->n_types || j >= c->n_types || i == j || !std::isfinite(chiN_ij))
        return fail(SOMA_EINVAL, "soma_set_chi: need 0 <= i != j < n_types and a finite value");
    c->chiN[i][j] = c->chiN[j][i] = chiN_ij;
    return refresh_fields(c);
}

int soma_set_external(soma_ctx* c, const float* ext_field, const uint8_t* forbidden, int src_is_device)
{
    if (!c) return fail(SOMA_EINVAL, "soma_set_external: ctx is NULL");
    DeviceGuard on_device(c->device);
    const cudaMemcpyKind kind = src_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    const size_t n = (size_t)c->cells * c->n_types;
    if (ext_field) {
        if (!c->ext) CU(cudaMalloc(&c->ext, sizeof(float) * n));
        CU(cudaMemcpyAsync(c->ext, ext_field, sizeof(float) * n, kind, c->stream));
    } else if (c->ext) {
        CU(cudaStreamSynchronize(c->stream));
        CU(cudaFree(c->ext));
        c->ext = nullptr;
    }
    c->n_forbidden = 0;
    if (forbidden) {
        if (!c->forbidden) CU(cudaMalloc(&c->forbidden, c->cells));
        CU(cudaMemcpyAsync(c->forbidden, forbidden, c->cells, kind, c->stream));
        // the accessible volume normalises phi: count the forbidden cells on the host (one byte per cell)
        std::vector<uint8_t> h(c->cells);
        CU(cudaMemcpyAsync(h.data(), c->forbidden, c->cells, cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
        for (uint8_t v : h) c->n_forbidden += v ? 1 : 0;
        if (c->n_forbidden >= c->cells) {
            c->n_forbidden = 0;
            CU(cudaFree(c->forbidden));
            c->forbidden = nullptr;
            return fail(SOMA_EINVAL, "soma_set_external: every cell is forbidden");
        }
    } else if (c->forbidden) {
        CU(cudaStreamSynchronize(c->stream));
        CU(cudaFree(c->forbidden));
        c->forbidden = nullptr;
    }
    int rc = refresh_fields(c);
    if (rc) return rc;
    if (!src_is_device) CU(cudaStreamSynchronize(c->stream));   // the caller may reuse its buffers
    return SOMA_OK;
}

int soma_set_option(soma_ctx* c, int key, double value)
{
    if (!c) return fail(SOMA_EINVAL, "soma_set_option: ctx is NULL");
    DeviceGuard on_device(c->device);
    const int iv = (int)value;
    switch (key) {
        case SOMA_OPT_HAMILTONIAN:
            if (iv != 0 && iv != 1) return fail(SOMA_EINVAL, "SOMA_OPT_HAMILTONIAN: 0 or 1");
            c->hamiltonian = iv;
            return refresh_fields(c);
        case SOMA_OPT_MOVE:
            if (iv != 1 && iv != 2) return fail(SOMA_EINVAL, "SOMA_OPT_MOVE: 1 (local) or 2 (Smart-MC)");
            c->move = iv;
            return SOMA_OK;
        case SOMA_OPT_SMC_STEP:
            if (!(value > 0.0) || !std::isfinite(value)) return fail(SOMA_EINVAL, "SOMA_OPT_SMC_STEP: must be > 0");
            // the proposal's Gaussians are off by up to ~2e-6 (draw_move), a displacement by sqrt(2 a_s) times
            // that: within the 1e-6 R_e0 this library states for Smart-MC positions only while sqrt(2 a_s) <= 0.5
            if (value > 0.125)
                return fail(SOMA_EINVAL, "SOMA_OPT_SMC_STEP: a_s must be <= 0.125 R_e0^2 (beyond it the approximate "
                            "Box-Muller of the proposal no longer keeps displacements within 1e-6 R_e0 of the exact ones)");
            c->smc_step = (float)value;
            return SOMA_OK;
        case SOMA_OPT_RECORD_DECISIONS:
            c->record = iv != 0;
            return SOMA_OK;
        case SOMA_OPT_KERNEL:
            if (iv < 0 || iv > 2) return fail(SOMA_EINVAL, "SOMA_OPT_KERNEL: 0, 1 or 2");
            if (iv == 2)
                for (const Spec& s : c->specs)
                    if (!s.fused_ok) return fail(SOMA_EINVAL, "SOMA_OPT_KERNEL=2: chain length %u cannot use the fused kernel", s.N);
            c->kernel_choice = iv;
            return SOMA_OK;
        case SOMA_OPT_DENSITY:
            if (iv != 0 && iv != 1) return fail(SOMA_EINVAL, "SOMA_OPT_DENSITY: 0 or 1");
            c->density_mode = iv;
            return SOMA_OK;
        case SOMA_OPT_TIMING: {
            int rc = drain_events(c);
            c->timing = iv != 0;
            return rc;
        }
        case SOMA_OPT_SWEEP_COUNTER:
            if (value < 0) return fail(SOMA_EINVAL, "SOMA_OPT_SWEEP_COUNTER: must be >= 0");
            c->sweep = (uint64_t)value;
            return SOMA_OK;
        case SOMA_OPT_PDL:
            if (iv != 0 && iv != 1) return fail(SOMA_EINVAL, "SOMA_OPT_PDL: 0 or 1");
            c->pdl = iv;
            return SOMA_OK;
        case SOMA_OPT_LAYOUT: {
            if (iv != 0 && iv != 1) return fail(SOMA_EINVAL, "SOMA_OPT_LAYOUT: 0 or 1");
            if (iv == c->layout) return SOMA_OK;
            if (iv == 1) {
                c->layout = 1;
                return resort(c);
            }
            // back to the caller's order: export, reset orig to the identity, import
            int rc = ensure_stage(c);
            if (rc) return rc;
            rc = copy_soa(c, c->stage, nullptr, true, true);
            if (rc) return rc;
            for (const Spec& s : c->specs)
                if (s.n_chains)
                    soma::iota_kernel<<<(unsigned)((s.n_chains + 255) / 256), 256, 0, c->stream>>>(c->orig + s.chain_off, (uint32_t)s.n_chains);
            c->layout = 0;
            return copy_soa(c, nullptr, c->stage, false, true);
        }
        case SOMA_OPT_SCHEME:
            if (iv != 0 && iv != 1) return fail(SOMA_EINVAL, "SOMA_OPT_SCHEME: 0 (independent sets) or 1 (molecule-parallel)");
            c->scheme = iv;
            return SOMA_OK;
        case SOMA_OPT_SET_ORDER:
            if (iv != 0 && iv != 1) return fail(SOMA_EINVAL, "SOMA_OPT_SET_ORDER: 0 (even, odd) or 1 (random per chain and sweep)");
            if (iv == 1 && c->kernel_choice == 2 && c->move == 2)
                return fail(SOMA_EINVAL, "SOMA_OPT_SET_ORDER=1 with Smart-MC needs the generic kernel (SOMA_OPT_KERNEL 0 or 1)");
            c->set_order = iv;
            return SOMA_OK;
        case SOMA_OPT_FIELD_INTERVAL:
            if (iv < 1) return fail(SOMA_EINVAL, "SOMA_OPT_FIELD_INTERVAL: must be >= 1");
            c->field_interval = iv;
            return SOMA_OK;
        case SOMA_OPT_COUNT_BITS: {
            if (iv != 0 && iv != 16 && iv != 32) return fail(SOMA_EINVAL, "SOMA_OPT_COUNT_BITS: 0 (auto), 16 or 32");
            if (iv == 16 && c->n_types != 2) return fail(SOMA_EINVAL, "SOMA_OPT_COUNT_BITS=16: the packed format holds two bead types");
            c->count_bits = iv;
            const bool want = want_pack(c);
            CU(cudaStreamSynchronize(c->stream));
            if (want == c->pack && !*(volatile uint32_t*)c->overflow_host) return SOMA_OK;
            // recount in the new format (the flag of an earlier overflow goes with the old counters)
            *(volatile uint32_t*)c->overflow_host = 0u;
            c->pack = want;
            int rc = upload_toff(c);
            if (rc) return rc;
            return stage1(c, "SOMA_OPT_COUNT_BITS");
        }
        case SOMA_OPT_SORT_INTERVAL:
            if (iv < 0) return fail(SOMA_EINVAL, "SOMA_OPT_SORT_INTERVAL: must be >= 0");
            c->sort_interval = iv;
            return SOMA_OK;
        default:
            return fail(SOMA_EINVAL, "soma_set_option: unknown key %d", key);
    }
}

int soma_stats(soma_ctx* c, uint64_t* attempted, uint64_t* accepted, uint64_t* sweeps_done)
{
    if (!c) return fail(SOMA_EINVAL, "soma_stats: ctx is NULL");
    DeviceGuard on_device(c->device);
    CU(cudaMemcpyAsync(c->acc_host, c->acc_slots, sizeof(unsigned long long) * soma::kAccSlots,
                       cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    uint64_t acc = 0;
    for (int i = 0; i < soma::kAccSlots; ++i) acc += c->acc_host[i];
    if (attempted) *attempted = c->attempted;
    if (accepted) *accepted = acc;
    if (sweeps_done) *sweeps_done = c->sweep;
    return check_overflow(c, "soma_stats");
}

int soma_decisions(soma_ctx* c, uint32_t* bits, int dst_is_device)
{
    if (!c || !bits) return fail(SOMA_EINVAL, "soma_decisions: NULL argument");
    DeviceGuard on_device(c->device);
    if (!c->decisions_valid)
        return fail(SOMA_ESTATE, "soma_decisions: set SOMA_OPT_RECORD_DECISIONS=1 before the sweep");
    CU(cudaMemcpyAsync(bits, c->decisions, sizeof(uint32_t) * ((c->n_beads_global + 31) / 32),
                       dst_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, c->stream));
    if (!dst_is_device) CU(cudaStreamSynchronize(c->stream));
    return SOMA_OK;
}

int soma_kernel_times(soma_ctx* c, double* ms, uint64_t* launches)
{
    if (!c) return fail(SOMA_EINVAL, "soma_kernel_times: ctx is NULL");
    DeviceGuard on_device(c->device);
    int rc = drain_events(c);
    if (rc) return rc;
    for (int k = 0; k < SOMA_K_COUNT; ++k) {
        if (ms) ms[k] = c->t_ms[k];
        if (launches) launches[k] = c->t_launches[k];
        c->t_ms[k] = 0.0;
        c->t_launches[k] = 0;
    }
    return SOMA_OK;
}

uint64_t soma_launch_count(const soma_ctx* c) { return c ? c->launches : 0; }
uint64_t soma_n_beads(const soma_ctx* c) { return c ? c->n_beads : 0; }
uint64_t soma_n_cells(const soma_ctx* c) { return c ? c->cells : 0; }
int soma_n_types(const soma_ctx* c) { return c ? c->n_types : 0; }

int soma_sync(soma_ctx* c)
{
    if (!c) return fail(SOMA_EINVAL, "soma_sync: ctx is NULL");
    DeviceGuard on_device(c->device);
    CU(cudaStreamSynchronize(c->stream));
    CU(cudaGetLastError());
    return check_overflow(c, "soma_sync");
}

}  // extern "C"

// ================================================================================================
// soma_fields_static: stage 1 of a configuration the caller holds, for callers that cannot allocate
// (include/soma_b200.h says who they are).  The occupation numbers -- the only memory stage 1 needs
// besides its input and output -- are a file-scope device array: part of the library image, 4 MiB on
// every GPU that has loaded this library, shared by every call.  Nothing above this line uses it, and
// nothing below calls cudaMalloc, cudaFree or a library routine that allocates.
// ================================================================================================
namespace {

constexpr uint32_t kStaticTail = 64;   // words behind the occupation numbers; word 0: beads outside the coordinate domain

// In HOST code this name is only a handle for cudaGetSymbolAddress (it is not a device address: a kernel
// handed `g_static_words` itself would read and write the wrong memory); device code may name it directly.
static __device__ __align__(256) uint32_t g_static_words[SOMA_STATIC_MAX_WORDS + kStaticTail];

struct StaticTypes {
    uint8_t t[SOMA_STATIC_MAX_MONOMERS];   // bead type per monomer, the architectures one after the other
};

// histogram_kernel<false> with the type table in the kernel's parameters instead of in device memory
// (a table in device memory would be one more buffer to allocate): Eq. 4, one count per bead.
__global__ void __launch_bounds__(256)
static_histogram_kernel(const soma::GridP g, const float* __restrict__ x, const float* __restrict__ y,
                        const float* __restrict__ z, const __grid_constant__ StaticTypes types, uint32_t first,
                        uint32_t N, uint32_t n_beads, uint32_t* __restrict__ counts, uint32_t* __restrict__ n_outside)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    uint32_t bad = 0;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_beads; i += stride) {
        const uint32_t j = (uint32_t)(i % N);
        const float xi = x[i], yi = y[i], zi = z[i];
        const uint32_t idx = soma::cell_at<false>(g, xi, yi, zi, (uint32_t)types.t[first + j] * g.cells + g.k_rec);
        atomicAdd(counts + idx, 1u);
        // the supported coordinates of cell_raw(): |t n| < 2^22 per axis (a NaN fails the comparison too)
        const bool ok = fabsf(xi * g.inv_L[0] * g.nf[0]) < 4194304.0f && fabsf(yi * g.inv_L[1] * g.nf[1]) < 4194304.0f &&
                        fabsf(zi * g.inv_L[2] * g.nf[2]) < 4194304.0f;
        bad += ok ? 0u : 1u;
    }
    if (bad) atomicAdd(n_outside, bad);
}

// Where the current device keeps g_static_words.  Looked up once per device, with that device current.
std::mutex g_static_mutex;
uint32_t* g_static_addr[kMaxDevices] = {};

int static_words_of(int dev, uint32_t** out)
{
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_addr[dev]) {
        void* p = nullptr;
        CU(cudaGetSymbolAddress(&p, g_static_words));
        if (!p) return fail(SOMA_ECUDA, "soma_fields_static: cudaGetSymbolAddress returned no address on device %d", dev);
        g_static_addr[dev] = static_cast<uint32_t*>(p);
    }
    *out = g_static_addr[dev];
    return SOMA_OK;
}

// Is p device memory of device dev?  (A host pointer here would fault in the kernel, or on a system where
// the GPU reaches host memory be used silently.)
int static_check_pointer(const void* p, int dev, const char* name)
{
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) {
        cudaGetLastError();
        return fail(SOMA_EINVAL, "soma_fields_static: %s is not a CUDA pointer", name);
    }
    if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged)
        return fail(SOMA_EINVAL, "soma_fields_static: %s must be device memory", name);
    if (at.type == cudaMemoryTypeDevice && at.device != dev)
        return fail(SOMA_EINVAL, "soma_fields_static: %s lives on device %d, the current device is %d", name, at.device, dev);
    return SOMA_OK;
}

}  // namespace

extern "C" int soma_fields_static(const soma_chain_spec* chains, int n_specs, int N_ref, int n_types, const float* box,
                                  const int* grid, float chiN, float kappaN, int hamiltonian, const float* dev_xyz,
                                  float* dev_omega, uint32_t* dev_counts, void* cuda_stream)
{
    // ---- arguments: everything that can be refused is refused before the device is touched
    if (!chains || n_specs < 1) return fail(SOMA_EINVAL, "soma_fields_static: need at least one chain spec");
    if (N_ref < 1) return fail(SOMA_EINVAL, "soma_fields_static: N_ref must be >= 1");
    if (n_types < 1 || n_types > SOMA_MAX_TYPES)
        return fail(SOMA_EINVAL, "soma_fields_static: n_types must be in 1..%d", SOMA_MAX_TYPES);
    if (!box || !grid) return fail(SOMA_EINVAL, "soma_fields_static: box/grid is NULL");
    if (hamiltonian != 0 && hamiltonian != 1) return fail(SOMA_EINVAL, "soma_fields_static: hamiltonian must be 0 or 1");
    if (!std::isfinite(chiN) || !std::isfinite(kappaN)) return fail(SOMA_EINVAL, "soma_fields_static: chiN/kappaN not finite");
    soma_ctx p;                       // host-side parameter block only: gridp() / fieldp() as the contexts compute them
    p.n_types = n_types;
    p.N_ref = N_ref;
    p.kappaN = kappaN;
    p.hamiltonian = hamiltonian;
    p.cells = 1;
    for (int a = 0; a < 3; ++a) {
        if (!(box[a] > 0.0f) || !std::isfinite(box[a])) return fail(SOMA_EINVAL, "soma_fields_static: box[%d] must be > 0", a);
        if (grid[a] < 1 || grid[a] > (1 << 22)) return fail(SOMA_EINVAL, "soma_fields_static: grid[%d] must be in 1..2^22", a);
        p.box[a] = box[a];
        p.grid[a] = grid[a];
        p.cells *= (uint64_t)grid[a];
        if (p.cells > SOMA_STATIC_MAX_WORDS) break;
    }
    const uint64_t words = p.cells * (uint64_t)n_types;
    if (p.cells > SOMA_STATIC_MAX_WORDS || words > SOMA_STATIC_MAX_WORDS)
        return fail(SOMA_EINVAL, "soma_fields_static: the grid needs more than the %u words (n_types * cells) of the "
                    "library's static array; larger grids need a context (soma_init), which allocates",
                    (unsigned)SOMA_STATIC_MAX_WORDS);
    for (int i = 0; i < n_types; ++i)
        for (int k = 0; k < n_types; ++k) p.chiN[i][k] = i == k ? 0.0f : chiN;
    StaticTypes types = {};
    uint64_t n_monomers = 0, n_beads = 0;
    for (int a = 0; a < n_specs; ++a) {
        const uint32_t N = chains[a].n_beads;
        if (N < 1 || (chains[a].n_chains > 0 && !chains[a].types))
            return fail(SOMA_EINVAL, "soma_fields_static: spec %d: n_beads must be >= 1 and types non-NULL", a);
        if (n_monomers + N > SOMA_STATIC_MAX_MONOMERS)
            return fail(SOMA_EINVAL, "soma_fields_static: the architectures have more than %u monomers in all; such "
                        "systems need a context (soma_init), which allocates", (unsigned)SOMA_STATIC_MAX_MONOMERS);
        for (uint32_t j = 0; j < N; ++j) {
            const uint8_t t = chains[a].n_chains ? chains[a].types[j] : 0;
            if (t >= n_types)
                return fail(SOMA_EINVAL, "soma_fields_static: spec %d monomer %u has type %u >= n_types", a, j, (unsigned)t);
            types.t[n_monomers + j] = t;
        }
        n_monomers += N;
        if (chains[a].n_chains >= (1ull << 32) || (n_beads += chains[a].n_chains * N) >= (1ull << 32))
            return fail(SOMA_EINVAL, "soma_fields_static: total beads must be < 2^32");
    }
    if (n_beads == 0) return fail(SOMA_EINVAL, "soma_fields_static: the system has no beads");
    if (!dev_xyz || !dev_omega) return fail(SOMA_EINVAL, "soma_fields_static: dev_xyz / dev_omega is NULL");
    p.n_beads = p.n_beads_global = n_beads;

    // ---- device
    int n_dev = 0, dev = 0, major = 0, n_sm = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev < 1) {
        cudaGetLastError();
        return fail(SOMA_ENODEVICE, "soma_fields_static: no CUDA device (this library has no CPU path)");
    }
    CU(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return fail(SOMA_EINVAL, "soma_fields_static: device %d is beyond the %d this library tracks", dev, kMaxDevices);
    CU(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    CU(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    if (major != 10) return fail(SOMA_ENODEVICE, "soma_fields_static: kernels are built for sm_100a only, device is sm_%dx", major);
    int rc = static_check_pointer(dev_xyz, dev, "dev_xyz");
    if (!rc) rc = static_check_pointer(dev_omega, dev, "dev_omega");
    if (!rc && dev_counts) rc = static_check_pointer(dev_counts, dev, "dev_counts");
    if (rc) return rc;
    uint32_t* words_dev = nullptr;    // the DEVICE address of g_static_words on this device
    rc = static_words_of(dev, &words_dev);
    if (rc) return rc;
    uint32_t* n_outside = words_dev + SOMA_STATIC_MAX_WORDS;
    cudaStream_t stream = (cudaStream_t)cuda_stream;

    // ---- a3: the array keeps the last call's numbers; clear what this call counts into
    CU(cudaMemsetAsync(words_dev, 0, sizeof(uint32_t) * words, stream));
    CU(cudaMemsetAsync(n_outside, 0, sizeof(uint32_t), stream));
    const soma::GridP g = p.gridp();
    uint64_t bead0 = 0;
    uint32_t first = 0;
    for (int a = 0; a < n_specs; ++a) {
        const uint32_t N = chains[a].n_beads;
        const uint64_t nb = chains[a].n_chains * N;
        if (nb) {
            const int threads = 256;
            const uint64_t blocks = std::min<uint64_t>((nb + threads - 1) / threads, (uint64_t)n_sm * 16);
            static_histogram_kernel<<<(unsigned)blocks, threads, 0, stream>>>(
                g, dev_xyz + bead0, dev_xyz + n_beads + bead0, dev_xyz + 2 * n_beads + bead0, types, first, N, (uint32_t)nb,
                words_dev, n_outside);
            CU(cudaGetLastError());
        }
        bead0 += nb;
        first += N;
    }

    // ---- a4: the contexts' field kernel, reading the static array, writing the caller's omega
    const soma::FieldP F = p.fieldp();
    const int threads = 256;
    const unsigned blocks = (unsigned)((p.cells + threads - 1) / threads);
    switch (n_types) {
        case 1: CU(launch_pdl(false, soma::field_kernel<1, false>, blocks, threads, 0, stream, F, words_dev, dev_omega, nullptr, nullptr, nullptr, nullptr, 0ull, nullptr, nullptr, 0u, (size_t)0)); break;
        case 2: CU(launch_pdl(false, soma::field_kernel<2, false>, blocks, threads, 0, stream, F, words_dev, dev_omega, nullptr, nullptr, nullptr, nullptr, 0ull, nullptr, nullptr, 0u, (size_t)0)); break;
        default: CU(launch_pdl(false, soma::field_kernel<0, false>, blocks, threads, 0, stream, F, words_dev, dev_omega, nullptr, nullptr, nullptr, nullptr, 0ull, nullptr, nullptr, 0u, (size_t)0)); break;
    }
    if (dev_counts) CU(cudaMemcpyAsync(dev_counts, words_dev, sizeof(uint32_t) * words, cudaMemcpyDeviceToDevice, stream));
    uint32_t bad = 0;
    CU(cudaMemcpyAsync(&bad, n_outside, sizeof(uint32_t), cudaMemcpyDeviceToHost, stream));
    CU(cudaStreamSynchronize(stream));
    if (bad)
        return fail(SOMA_EDOMAIN, "soma_fields_static: %u beads have a coordinate that is not finite or lies outside "
                    "the supported domain |x n / L| < 2^22 per axis", bad);
    return SOMA_OK;
}
