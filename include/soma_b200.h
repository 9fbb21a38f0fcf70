/*
 * soma_b200.h -- C ABI of the B200-native SCMF Monte-Carlo step (SOMA, arXiv:1711.03828).
 *
 * One SCMF cycle ("MC step") as this library runs it:
 *     a1  local-displacement Metropolis moves of the even monomers of every chain   (Eq. 2, Eq. 15)
 *     a2  the same for the odd monomers (independent sets of Fig. 1 / Code 2)
 *     a3  occupation numbers n_i(c), Eq. 4
 *     a4  interaction fields omega_i(c), Eq. 12
 * with the fields frozen during a1/a2.  a5 (Smart-MC) replaces a1/a2 on request.
 * Every step runs in CUDA kernels written for sm_100a; there is no CPU fallback.
 *
 * Conventions
 *   - plain C, no exceptions cross the boundary; every int-returning call gives SOMA_OK (0) or a
 *     negative SOMA_E* code and leaves a message for soma_last_error() (thread-local).
 *   - lengths are in units of R_e0; energies in k_B T.
 *   - bead arrays are chain-major SoA float32: xyz = x[n_beads] | y[n_beads] | z[n_beads], bead
 *     index = (beads of earlier architectures) + chain * n_beads_per_chain + monomer; coordinates
 *     are unwrapped (never folded into the box).
 *   - grid arrays are [type][ix][iy][iz], iz fastest; cell (ix,iy,iz) is the half-open box
 *     [ix dLx,(ix+1) dLx) x ... that *contains* the bead (Pi_c of Eq. 4), periodic images folded:
 *     per axis t = fl32(x * fl32(1/L)), cell = floor(t n) mod n in exact arithmetic (R7).
 *     Supported coordinates: |t n| < 2^22 per axis (at least 2^22 / n box lengths from the origin in
 *     either direction); outside of it, and for NaN, the cell is unspecified but always a valid index.
 *   - pointers named host_* are host memory, dev_* device memory; "dst_is_device" selects.
 *   - the library owns all device state of a context; callers own every buffer they pass in; input
 *     buffers are only read during the call.
 *   - all work is enqueued on the CUDA stream given to soma_init (NULL = legacy default stream);
 *     calls that write host memory synchronise that stream before returning, soma_step does not.
 *   - random numbers: Philox4x32-10, counter = (global bead index, sweep lo32, sweep hi32,
 *     (kind << 8) | sub), key = (seed lo32, seed hi32); kind 0 initial state, 1 local move,
 *     2 Smart-MC.  Results depend on (seed, sweep counter, positions) only.
 */
#ifndef SOMA_B200_H
#define SOMA_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SOMA_MAX_TYPES 8

enum {
    SOMA_OK = 0,
    SOMA_EINVAL = -1,    /* bad argument (message says which)                 */
    SOMA_ECUDA = -2,     /* a CUDA runtime call or kernel failed              */
    SOMA_ENOMEM = -3,    /* device or host allocation failed                  */
    SOMA_ESTATE = -4,    /* call not valid in the current state of the context */
    SOMA_ENODEVICE = -5, /* no CUDA device / wrong architecture (needs sm_100) */
    SOMA_EDOMAIN = -6,   /* a coordinate handed in is NaN / infinite / outside |x n / L| < 2^22 */
    SOMA_EOVERFLOW = -7  /* a cell holds more than 65535 beads of one type while the occupation numbers are
                            kept as 16 + 16 bits per cell (SOMA_OPT_COUNT_BITS).  Sticky: the field kernel sets
                            it on the device; soma_step (on entry), soma_sync, soma_stats and the calls that
                            copy to host memory report it from then on.  Fields and trajectory are invalid
                            from the sweep in which it happened: set SOMA_OPT_COUNT_BITS = 32 and go back to a
                            saved configuration (soma_set_positions)                                  */
};

/* keys of soma_set_option */
enum {
    SOMA_OPT_HAMILTONIAN = 1,      /* 0: K^0_inter (Eq. 7, default), 1: K^1_inter (Eq. 8); refreshes omega   */
    SOMA_OPT_MOVE = 2,             /* 1: local displacement (default), 2: Smart-MC                            */
    SOMA_OPT_SMC_STEP = 3,         /* Smart-MC step a_s in R_e0^2, 0 < a_s <= 0.125 (SOMA_EINVAL beyond: the  */
                                   /* proposal's fast Box-Muller is accurate to ~2e-6 per Gaussian, so that a  */
                                   /* displacement stays within 1e-6 R_e0 of the exact one up to sqrt(2 a_s) = 0.5) */
    SOMA_OPT_RECORD_DECISIONS = 4, /* 1: keep the accept/reject bit of every move of the last sweep           */
    SOMA_OPT_KERNEL = 5,           /* 0: auto (default); 1: force the one-thread-per-monomer kernels on global */
                                   /* memory (two launches per sweep for linear chains, one per independent   */
                                   /* set for bond-list architectures, no shared-memory staging);              */
                                   /* 2: chain-resident fused kernel (error if an architecture cannot use it:  */
                                   /* it takes linear chains whose length is a multiple of 4 and at most 128)  */
    SOMA_OPT_DENSITY = 6,          /* 0: incremental count update fused into the move kernel (default),       */
                                   /* 1: clear + full histogram kernel after every sweep                      */
    SOMA_OPT_TIMING = 7,           /* 1: bracket every kernel with CUDA events (see soma_kernel_times)        */
    SOMA_OPT_SWEEP_COUNTER = 8,    /* set the sweep counter (the "time step" word of the Philox counter)      */
                                   /* (keys 9 and 10 are not used)                                             */
    SOMA_OPT_LAYOUT = 11,          /* 0: chains stay in the caller's order in device memory; 1 (default): the  */
                                   /* library keeps them in Hilbert order of their centres of mass.  Storage   */
                                   /* only: every result is identical, every API array is in the caller's order */
    SOMA_OPT_SORT_INTERVAL = 12,   /* re-sort every this many sweeps (default 2000; 0: only at init/set_positions) */
    SOMA_OPT_SET_ORDER = 13,       /* 0 (default): even monomers, then odd monomers, every sweep; 1: the order */
                                   /* of the two sets is drawn per chain and sweep ("random permutation of the */
                                   /* sets", Code 2): Philox kind 3, counter word 0 = global */
                                   /* index of the chain's first bead, bit 31 of word 0, 1 = odd set first     */
    SOMA_OPT_FIELD_INTERVAL = 14,  /* k >= 1 (default 1): omega is refreshed after sweeps number k, 2k, ...    */
                                   /* (counted from 1); the occupation numbers are current after every sweep   */
    SOMA_OPT_SCHEME = 15,          /* 0 (default): independent sets, every particle attempted exactly once per */
                                   /* sweep (Code 2); 1: molecule-parallel scheme (Code 1):   */
                                   /* every molecule picks N times one of its particles at random.  Attempt k  */
                                   /* of the chain whose first bead is f uses Philox counter word f + k: kind 4 */
                                   /* word 0 picks i = floor(w N / 2^32), kinds 1 / 2 drive the move; bit f + k */
                                   /* of soma_decisions is the outcome of that attempt                          */
    SOMA_OPT_PDL = 16,             /* 1 (default): the fused move kernel and the field kernel are launched with */
                                   /* programmatic dependent launch, so each becomes resident while its         */
                                   /* predecessor drains (results do not depend on it); 0: ordinary launches    */
    SOMA_OPT_COUNT_BITS = 17       /* format of the grid arrays in device memory (storage only: soma_fields     */
                                   /* always returns [type][cell] arrays with uint32 occupation numbers).  32:  */
                                   /* planes omega[type][cell], uint32 n[type][cell].  16 (n_types = 2 only):   */
                                   /* one record {omega_A, omega_B} per cell and both occupation numbers in one */
                                   /* 32-bit word, 16 bits each, as PAPER.md:243 stores them (uint16): 12       */
                                   /* instead of 16 bytes per cell; a cell with more than 65535 beads of one    */
                                   /* type is detected whenever the fields are computed -> SOMA_EOVERFLOW.      */
                                   /* 0 (default): 16 if n_types = 2 and the planes would take more than 48 MB  */
                                   /* (they no longer stay in L2 beside the positions streaming through), else  */
                                   /* 32; soma_init and soma_set_positions fall back to 32 on their own if the  */
                                   /* configuration handed in is too dense (an overflow during later sweeps is  */
                                   /* reported, not repaired).  Recounts.                                        */
};

/* indices of soma_kernel_times */
enum { SOMA_K_MOVE = 0, SOMA_K_DENSITY = 1, SOMA_K_FIELD = 2, SOMA_K_LAYOUT = 3, SOMA_K_COUNT = 4 };

typedef struct soma_ctx soma_ctx; /* opaque */

/* One molecular architecture: n_chains molecules of n_beads monomers with the given bead types
 * (architecture stored once per molecule type).  n_bonds = 0: a linear chain
 * (monomer j bonded to j + 1).  n_bonds > 0: any architecture (stars, rings, ...) given by its bond
 * list; every bond is the harmonic spring of Eq. 2.  The library then builds the independent sets
 * by greedy first fit in monomer order -- monomer j joins the lowest-numbered set that
 * holds none of its bonded neighbours -- works through them in the order 0, 1, ..., and sums the
 * bonds of a monomer in ascending order of the neighbour's index (R25).  Architectures
 * with a bond list support SOMA_OPT_SCHEME 0 and SOMA_OPT_SET_ORDER 0 only. */
typedef struct {
    uint64_t        n_chains;
    uint32_t        n_beads;
    const uint8_t  *types;   /* host, [n_beads], each < n_types; read during soma_init only          */
    uint32_t        n_bonds; /* 0: linear chain                                                       */
    const uint32_t *bonds;   /* host, [2 * n_bonds] monomer pairs (i, j), i != j, each pair once; or NULL */
} soma_chain_spec;

/* The architecture array the library keeps for a molecule type given by a bond list: the 32-bit words of Fig. 2
 * -- word 0: N; words 1..N, per monomer: (index of its first bond word << 8) | type, index 0 if it
 * has no bond; then per bond, in ascending order of the partner: (signed offset to the partner << 5) | (bond type
 * << 1) | 1 on the monomer's last bond -- followed by the independent sets (greedy first fit):
 * members[N] set by set | set_off[n_sets + 1] | floor(2^32 / set size) + 1 per set.  Host only (no device needed):
 * for inspection and tests.  words_out may be NULL to ask for the length; *n_sets (nullable) gets the number of sets. */
int soma_architecture_words(const soma_chain_spec *spec, uint32_t *words_out, uint64_t capacity, uint64_t *n_words,
                            uint32_t *n_sets);

/* Create a system and run stage 1 (densities, fields) on its initial configuration.
 *   chains/n_specs  architectures, stored one after the other in the bead arrays (n_specs >= 1)
 *   N_ref           reference chain length N of PAPER.md:157: k_0 = 3 (N_ref-1)/R_e0^2 (Eq. 2 with
 *                   b_0 = sqrt(3/k_0)), chi_0 = chiN/N_ref, kappa_0 = kappaN/N_ref
 *   n_types         bead types n_t, 1..SOMA_MAX_TYPES
 *   box, grid       periodic box lengths and cells per axis (host, 3 values each)
 *   chiN            Flory-Huggins chi N used for every unordered type pair (see soma_set_chi)
 *   kappaN          Helfand compressibility kappa N (Eq. 6)
 *   A               maximal step length a of the local move; 0 < A <= min(box)/2
 *   seed            Philox key
 *   host_xyz0       initial positions (host, SoA 3*n_beads floats) or NULL: the library then draws
 *                   Gaussian random walks (first bead uniform in the box, per-axis bond std
 *                   R_e0/sqrt(3 (N_ref-1))) from kind-0 Philox words on the device
 *   cuda_stream     cudaStream_t to run on (e.g. torch.cuda.current_stream().cuda_stream) or NULL
 * Total beads must be < 2^32 (the bead index is one Philox counter word), cells < 2^31. */
int soma_init(soma_ctx **out, const soma_chain_spec *chains, int n_specs, int N_ref, int n_types,
              const float *box, const int *grid, float chiN, float kappaN, float A, uint64_t seed,
              const float *host_xyz0, void *cuda_stream);

/* Several GPUs ("molecules are distributed among the MPI ranks", every rank keeps the
 * whole grid, the densities are summed over the ranks after every MC step).  A rank
 * creates a context from its own molecules and says where they sit in the whole system:
 *   spec_first_bead  host, [n_specs]: index, in the whole system's bead numbering, of the first bead of
 *                    this rank's molecules of each architecture.  It is the Philox counter word of that
 *                    bead, so a shard draws exactly the numbers the undivided system draws for these
 *                    molecules (and the decision bitmap is indexed by it: soma_decisions then returns
 *                    ceil(global_n_beads / 32) words)
 *   global_n_beads   beads of the whole system (< 2^32): rho_0 of Eq. 12 is global_n_beads / volume
 * All other arguments as for soma_init, describing this rank's molecules only (host_xyz0: their
 * positions, or NULL to draw them as the undivided system would).
 *
 * The exchange array.  A shard keeps two arrays of occupation numbers in the grid format of the context
 * (SOMA_OPT_COUNT_BITS): its copy of the WHOLE system's numbers (what soma_fields returns), and the exchange
 * array, into which its own kernels count -- the histogram of its molecules after soma_init_shard /
 * soma_set_positions, the +1 / -1 of its accepted moves after soma_shard_moves.  The caller sums the exchange
 * arrays of all ranks element-wise as uint32 (modulo 2^32; in place, any collective: NCCL all-reduce on the
 * device address soma_shard_exchange returns) and calls soma_shard_fields, whose kernel adds the sum to the
 * whole system's numbers, clears the exchange array for the next sweep and computes omega.  So per MC step:
 *     soma_shard_moves;  all-reduce (sum) of the exchange array;  soma_shard_fields(ctx, 1)
 * and once after soma_init_shard (or after every rank's soma_set_positions): all-reduce; soma_shard_fields(ctx, 0).
 * No copy and no conversion lies between the move kernel, the collective and the field kernel.  The
 * positions, occupation numbers and fields equal those of the undivided system bit for bit.  soma_step
 * returns SOMA_ESTATE on such a context.  Every rank must use the same grid format: a shard does not fall
 * back from the packed records on its own (an overflow shows as SOMA_EOVERFLOW after the next
 * soma_shard_fields), and after SOMA_OPT_COUNT_BITS was changed -- on every rank -- the exchange array holds
 * the rank's histogram again and wants the all-reduce and soma_shard_fields(ctx, 0) like after soma_init_shard. */
int soma_init_shard(soma_ctx **out, const soma_chain_spec *chains, int n_specs, int N_ref, int n_types,
                    const float *box, const int *grid, float chiN, float kappaN, float A, uint64_t seed,
                    const float *host_xyz0, void *cuda_stream, const uint64_t *spec_first_bead,
                    uint64_t global_n_beads);

/* The moves of one sweep (a1, a2 | a5) of this rank's molecules in the current omega; the local
 * occupation numbers follow (a3).  Asynchronous on the context's stream.  SOMA_ESTATE for the
 * combinations whose part-of-a-system mode has no oracle: SOMA_OPT_SCHEME 1 and bond-list architectures. */
int soma_shard_moves(soma_ctx *ctx);

/* Device address and length (uint32 words) of the exchange array: n_types * cells words for planes, cells
 * words for the packed records.  Valid for the life of the context unless SOMA_OPT_COUNT_BITS is changed. */
int soma_shard_exchange(soma_ctx *ctx, void **dev_words, uint64_t *n_words);

/* The same array through host memory, for callers that sum on the host: to_host != 0 copies it out,
 * to_host = 0 copies host_words in.  Synchronises. */
int soma_shard_exchange_copy(soma_ctx *ctx, uint32_t *host_words, int to_host);

/* Peer mode: the field kernel does the reduction itself.  Instead of the caller's all-reduce, the kernel launched by
 * soma_shard_fields reads the exchange arrays of ALL ranks word by word through peer memory -- the other GPUs'
 * memory over NVLink / NVSwitch, mapped with CUDA IPC (or plain device addresses when the ranks are contexts of one
 * process) -- adds them up, folds the sum into the whole system's occupation numbers and computes omega: one kernel
 * for the exchange step and a4.  What remains for the caller is a BARRIER between soma_shard_moves and
 * soma_shard_fields (every rank's move kernel must have finished before any rank's field kernel reads its array;
 * in stream order, e.g. a one-element all-reduce enqueued behind the moves).  The exchange allocation holds two
 * buffers used alternately: the arrays a field kernel has read are left untouched (other ranks read them too) and
 * this rank's other buffer -- which every rank finished reading a sweep ago, by the same barrier -- is cleared for
 * the next sweep.  soma_shard_exchange then returns the buffer the NEXT soma_shard_moves counts into.
 *   soma_shard_peer_handle   64 bytes: the CUDA IPC handle of this rank's exchange allocation, to be sent to the peers
 *   soma_shard_set_peers     n_ranks, my_rank, and for every other rank either peer_dev[r] (device address of its
 *                            allocation = what soma_shard_exchange returned right after soma_init_shard; same
 *                            process) or, where that is NULL, handles[64 r .. 64 r + 63] (opened here).  Call it on
 *                            every rank after soma_init_shard and before the first soma_shard_fields.
 * Needs SOMA_OPT_FIELD_INTERVAL = 1 and the same SOMA_OPT_COUNT_BITS on every rank. */
int soma_shard_peer_handle(soma_ctx *ctx, void *handle64);
int soma_shard_set_peers(soma_ctx *ctx, int n_ranks, int my_rank, void *const *peer_dev, const void *handles);

/* a4: folds the (summed) exchange array into the whole system's occupation numbers, clears it, and computes
 * omega.  advance != 0 closes the sweep begun by soma_shard_moves (sweep counter + 1; omega is only
 * recomputed when SOMA_OPT_FIELD_INTERVAL says so, the numbers are folded in any case); advance = 0: stage 1
 * after soma_init_shard or soma_set_positions.  Launched with programmatic dependent launch (SOMA_OPT_PDL)
 * behind whatever precedes it in the stream. */
int soma_shard_fields(soma_ctx *ctx, int advance);

/* n_sweeps SCMF cycles: (a1, a2 | a5), a3, a4 each.  Asynchronous on the context's stream.
 * The sweep counter advances by n_sweeps. */
int soma_step(soma_ctx *ctx, int n_sweeps);

/* Copy out omega (float32 [n_types][cells]) and, if counts != NULL, the occupation numbers
 * (uint32 [n_types][cells]) that belong to the current positions. */
int soma_fields(soma_ctx *ctx, float *omega, uint32_t *counts, int dst_is_device);

/* Copy out the positions (SoA, 3*n_beads float32, unwrapped). */
int soma_positions(soma_ctx *ctx, float *xyz, int dst_is_device);

/* Replace the positions (SoA, 3*n_beads float32) and redo stage 1 (histogram + fields).  Synchronises.
 * SOMA_EDOMAIN if a coordinate is not finite or outside the supported domain (the positions are then
 * loaded all the same and the context stays usable, e.g. for another soma_set_positions); soma_init
 * returns the same code for its host_xyz0 and creates no context. */
int soma_set_positions(soma_ctx *ctx, const float *xyz, int src_is_device);

/* Set chi_ij N = chi_ji N for one type pair (i != j) and refresh omega. */
int soma_set_chi(soma_ctx *ctx, int i, int j, float chiN_ij);

/* External fields.  ext_field: float32 [n_types][cells], a static field added to
 * omega_i(c) ("a linear attraction for the particle of a specific type"), or NULL for none.
 * forbidden: uint8 [cells], non-zero = no particle may enter that cell ("geometric confinements"), or
 * NULL for none: omega is +inf there for every type, so every move into such a cell is rejected, and
 * phi_i is normalised with the accessible volume, rho_0 DeltaL^3 = beads / (cells - forbidden cells).
 * Beads that already sit in a forbidden cell are not moved out by this call (they may leave, never
 * return).  Both arrays are copied; omega is refreshed.  SOMA_EINVAL if every cell is forbidden. */
int soma_set_external(soma_ctx *ctx, const float *ext_field, const uint8_t *forbidden, int src_is_device);

int soma_set_option(soma_ctx *ctx, int key, double value);

/* attempted / accepted moves since soma_init and the current sweep counter (synchronises). */
int soma_stats(soma_ctx *ctx, uint64_t *attempted, uint64_t *accepted, uint64_t *sweeps_done);

/* Accept/reject bits of the last sweep, bit (b & 31) of word (b >> 5) for bead b, ceil(n_beads/32)
 * words; needs SOMA_OPT_RECORD_DECISIONS = 1 before that sweep. */
int soma_decisions(soma_ctx *ctx, uint32_t *bits, int dst_is_device);

/* Accumulated device time (ms) and launch count per kernel class since the last call; needs
 * SOMA_OPT_TIMING = 1.  Arrays of SOMA_K_COUNT entries (host).  Synchronises. */
int soma_kernel_times(soma_ctx *ctx, double *ms, uint64_t *launches);

/* Number of kernels this library has launched for ctx since soma_init (no synchronisation). */
uint64_t soma_launch_count(const soma_ctx *ctx);

/* n_beads / n_cells / n_types of a context (0 if ctx is NULL). */
uint64_t soma_n_beads(const soma_ctx *ctx);
uint64_t soma_n_cells(const soma_ctx *ctx);
int      soma_n_types(const soma_ctx *ctx);

/* Block until everything enqueued for ctx has finished. */
int soma_sync(soma_ctx *ctx);

void soma_destroy(soma_ctx *ctx);

/* Stage 1 (a3 + a4: occupation numbers of Eq. 4, then omega of Eq. 12) of a
 * configuration the CALLER holds in device memory, without a context and without a single allocation.
 *
 * Who this is for.  Every other entry point works on a soma_ctx, and soma_init pays for that context with
 * cudaMalloc.  Some programs that want the fields of a configuration cannot afford that call at the point where
 * they need them:
 *   - an analysis or steering tool that runs next to simulations which already fill the GPU (C4 alone is sized
 *     for the 180 GB): a cudaMalloc there fails, or succeeds only by making a caching allocator give memory back;
 *   - a host program (PyTorch is the usual case) whose allocator owns the device memory and hands out pieces of
 *     it: memory taken behind its back is invisible to its accounting, and it can lend this call buffers but not
 *     the right to allocate;
 *   - a loop that other streams run beside: cudaMalloc and cudaFree may wait for the whole device, so that one
 *     allocation in the wrong place stalls kernels that have nothing to do with this call.
 * For them the occupation numbers -- the only memory stage 1 needs besides its input and output -- live in an
 * array that is part of the library image: SOMA_STATIC_MAX_WORDS 32-bit words (4 MiB, plus a few counters) of
 * device memory on every GPU on which this library has been used, from the first use until the process exits,
 * whether or not this function is ever called again.  That is the price, and the limit: a grid with
 * n_types * cells > SOMA_STATIC_MAX_WORDS (C1, C2, C3 fit; C4 and C5 do not), or architectures with more than
 * SOMA_STATIC_MAX_MONOMERS monomers in all, are refused with SOMA_EINVAL before anything is launched.
 *
 *   chains/n_specs   as for soma_init (bond lists are ignored: bonds do not enter the densities); types are host
 *                    memory, read during the call
 *   N_ref, n_types, box, grid, chiN, kappaN   as for soma_init; hamiltonian as SOMA_OPT_HAMILTONIAN (0 | 1)
 *   dev_xyz          DEVICE, input: x[n] | y[n] | z[n] float32 of all n = sum n_chains * n_beads beads, the layout
 *                    of soma_positions
 *   dev_omega        DEVICE, output: float32 [n_types][cells]
 *   dev_counts       DEVICE, output, or NULL: uint32 [n_types][cells] occupation numbers
 *   cuda_stream      the stream the work is enqueued on (NULL: the legacy default stream)
 * Works on the calling thread's current device, which must own all three buffers.  The results equal, bit for bit,
 * what soma_fields returns from a context created by soma_init on the same positions with SOMA_OPT_COUNT_BITS = 32
 * (the same kernels' arithmetic; no external field, every type pair at chiN).
 *
 * No cudaMalloc, cudaFree or other allocating routine is called.  The first call on a device looks up where that
 * device keeps the array (cudaGetSymbolAddress, which makes the CUDA runtime load this library's kernels onto the
 * device if nothing has yet); later calls on that device reuse the address.  Make that first call before any
 * stream capture is begun.  The call synchronises cuda_stream before it returns (it reads back the counter of
 * out-of-domain coordinates): SOMA_EDOMAIN as for soma_set_positions, with omega and counts written all the same.
 *
 * One array per device serves every call, from every thread, on every stream, and keeps what the last call left
 * in it; each call clears the part it uses first.  Two calls that run on the same GPU at the same time therefore
 * corrupt each other's occupation numbers: callers serialise them (one stream, or their own ordering). */
#define SOMA_STATIC_MAX_WORDS    1048576u  /* n_types * cells                         */
#define SOMA_STATIC_MAX_MONOMERS 256u      /* monomers of all architectures together  */
int soma_fields_static(const soma_chain_spec *chains, int n_specs, int N_ref, int n_types, const float *box,
                       const int *grid, float chiN, float kappaN, int hamiltonian, const float *dev_xyz,
                       float *dev_omega, uint32_t *dev_counts, void *cuda_stream);

const char *soma_last_error(void);
const char *soma_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SOMA_B200_H */
