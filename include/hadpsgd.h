/*
 * hadpsgd.h -- C ABI of libhadpsgd.so: the per-step super-learner update of
 * Hierarchical ADPSGD (arxiv 1907.05701), emulated on one B200 (sm_100a).
 *
 * One call of hadpsgd_step() performs, for every super-learner s of S, every
 * parameter i of P, in ONE kernel launch and ONE pass over HBM:
 *   a2  gbar_s[i] = (1/G) * sum_{g<G} grad_{s,g}[i]        PAPER.md:57 eq. (6), :38 eq. (4), :84 (section 4)
 *   a3  v_s[i]    = mu * v_s[i] + gbar_s[i]                PAPER.md:34 eq. (3) + momentum (R2)
 *       u_s[i]    = w_s[i] - lr * v_s[i]
 *   a4  w_s[i]    = w_p[i] = 1/2 (u_s[i] + u_p[i])         PAPER.md:64-66 eq. (7), T_k; order per :62 (R3)
 *   a5  diagnostics: sum gbar^2, sum w'^2, sum (u_s-u_p)^2 PAPER.md:72 (consensus)
 * where p = partner(s, step_k) is the ring neighbour chosen by the pairing
 * scheduler (a1): even step_k pairs (2i,2i+1), odd pairs (2i+1,(2i+2) mod S).
 *
 * Conventions
 *  - Every function returns an int status: HADPSGD_OK (0) or a negative code.
 *    No exception crosses this boundary.  Nothing here falls back to the CPU.
 *  - "dev" pointers are DEVICE pointers, "host" pointers are HOST pointers.
 *  - The handle owns all descriptor memory.  Device memory is the caller's
 *    arena when opts->arena != NULL (never freed by the library), else owned
 *    by the library.  Pointers returned by weights/momentum/grads are
 *    borrowed and stay valid until hadpsgd_destroy().
 *  - hadpsgd_step() only enqueues work on the create-time stream and returns.
 *  - Layout: every buffer (S weight, S momentum, S*G gradient buffers) holds
 *    P_padded elements; segment k of the caller's table starts at an element
 *    offset that is a multiple of HADPSGD_SEG_ALIGN_ELEMS in every buffer;
 *    padding elements are zero at create and stay zero (zero gradient, zero
 *    weight, zero momentum), so they never perturb results or diagnostics.
 *    The caller must not write non-zero values into gradient padding.
 */
#ifndef HADPSGD_H
#define HADPSGD_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hadpsgd_ctx* hadpsgd_handle; /* opaque */

enum { HADPSGD_F32 = 0, HADPSGD_BF16 = 1 };

enum { /* status codes */
    HADPSGD_OK = 0,
    HADPSGD_INVALID_ARG = -1,        /* S<1, S>HADPSGD_MAX_S, G<1, n_seg<1, seg_len<1, bad dtype, index out
                                        of range, NULL out-pointer, a partner[] that is not a matching;
                                        hadpsgd_step with S odd and >1 (no perfect ring matching)      */
    HADPSGD_OUT_OF_MEMORY = -2,      /* arena too small / cudaMalloc failed                                */
    HADPSGD_CUDA = -3,               /* CUDA runtime or launch error; text via hadpsgd_last_error()        */
    HADPSGD_UNSUPPORTED_DEVICE = -4, /* compute capability != 10.x: no multi-backend dispatch, no fallback */
    HADPSGD_DIAG_TIMEOUT = -5        /* hadpsgd_diagnostics only: see "Sharing the device" there          */
};

enum { /* hadpsgd_opts.flags */
    HADPSGD_DETERMINISTIC = 1u << 0, /* one rounding per fp32 op, no FMA contraction, learners summed
                                        g=0..G-1: w and v are BIT-EXACT against the oracle               */
    HADPSGD_NO_MIX        = 1u << 1, /* T_k = I: eq. (6)/(3) only, every super-learner keeps u_s         */
    HADPSGD_NO_DIAG       = 1u << 2, /* skip a5                                                          */
    HADPSGD_EQ7_LITERAL   = 1u << 3, /* eq. (7) as printed: w'_s = 1/2 (w_s + w_p) - lr v_s  (row f1)    */
    HADPSGD_SHARE_PAIR_WEIGHTS = 1u << 4, /* both members of a pair end a step with identical weights (R3),
                                        so they SHARE one of the S weight buffers: one weight write per
                                        pair instead of two, and the buffer two neighbouring pairs read
                                        next step is fetched from HBM once.  Same arithmetic, same
                                        results; what changes is which buffer hadpsgd_weights(h, s)
                                        points to (see there).  Not with NO_MIX or EQ7_LITERAL.          */
    HADPSGD_PEER = 1u << 5           /* this handle holds the super-learners of ONE rank of a super-learner
                                        partition (row f4): see "super-learner partition"
                                        below.  Needs dtypes.peer_stage = 1.  Not with EQ7_LITERAL,
                                        SHARE_PAIR_WEIGHTS or a bf16 working copy.                        */
};

#define HADPSGD_SEG_ALIGN_ELEMS 64 /* 256 B in fp32, 128 B in bf16 */
#define HADPSGD_MAX_S 512

typedef struct {
    int32_t grad_dtype;   /* HADPSGD_F32 | HADPSGD_BF16 : dtype of the S*G learner gradient buffers */
    int32_t master_dtype; /* must be HADPSGD_F32 : weights AND momentum                             */
    int32_t working_dtype;/* HADPSGD_F32 (0, default): learners read the fp32 master weights, nothing
                             extra is stored.  HADPSGD_BF16: every step ALSO writes a bf16
                             (round-to-nearest-even) copy of each new weight buffer for
                             mixed-precision learners (+2 B per parameter per super-learner; row f2) */
    int32_t peer_stage;   /* 0 (default) | 1: also lay out two fp32 STAGE buffers per super-learner behind
                             the S weight buffers (+8 B per parameter per super-learner), in which the
                             halves of a mix between two arenas wait; required by HADPSGD_PEER          */
} hadpsgd_dtypes;

typedef struct {
    void*    arena;       /* dev; optional caller-owned memory (e.g. a torch uint8 tensor), 256 B aligned */
    size_t   arena_bytes; /* >= hadpsgd_required_bytes()                                                   */
    void*    stream;      /* cudaStream_t; NULL = the legacy default stream                                */
    uint32_t flags;       /* HADPSGD_DETERMINISTIC | NO_MIX | NO_DIAG | EQ7_LITERAL | SHARE_PAIR_WEIGHTS | PEER */
    int32_t  device;      /* CUDA device ordinal; -1 = current device                                      */
} hadpsgd_opts;

typedef struct { /* host-side copy of the a5 diagnostics of the most recent step */
    int32_t  S;
    int32_t  n_pairs;
    uint64_t step_k;
    double   gsq[HADPSGD_MAX_S]; /* sum_i gbar_s[i]^2                                  */
    double   wsq[HADPSGD_MAX_S]; /* sum_i w'_s[i]^2                                    */
    double   gap[HADPSGD_MAX_S]; /* sum_i (a_s[i]-a_p[i])^2 over the two vectors the mix averages (u; the old
                                    w under EQ7_LITERAL); gap[s]==gap[p]; exactly 0 if unmixed (R14) */
    /* HADPSGD_PEER only (all zero otherwise).  A member whose partner lives in another arena cannot
     * finish its mix inside this step: it reports wsq[s] = sum u_s^2, gap[s] = 0 and pending[s] = 1.
     * The launch that resolves the mix (the next step, or hadpsgd_peer_flush) then delivers what that
     * step still owed: pend_wsq[s] = sum_i w'_s[i]^2 and pend_gap[s] = sum_i (u_s[i]-u_p[i])^2.       */
    double   pend_wsq[HADPSGD_MAX_S];
    double   pend_gap[HADPSGD_MAX_S];
    int32_t  pending[HADPSGD_MAX_S]; /* after the most recent step: 1 = the mix of s awaits its partner   */
} hadpsgd_diag;

/* a0 replica allocator (host only, no GPU needed) ------------------------------------------- */

/* Bytes of device memory hadpsgd_create() needs for this configuration. */
int hadpsgd_required_bytes(int S, int G, const int64_t* seg_len /*host [n_seg]*/, int n_seg,
                           hadpsgd_dtypes dt, size_t* out_bytes);

/* The layout the allocator computes: element offset of every segment inside a buffer
 * (host out [n_seg], may be NULL), padded buffer length in elements, and byte offsets of
 * the weight, momentum and gradient regions inside the arena (each may be NULL).
 * weight buffer s   = arena + w_off + s * P_padded * 4
 * momentum buffer s = arena + v_off + s * P_padded * 4
 * gradient (s,g)    = arena + g_off + (s*G + g) * P_padded * sizeof(grad_dtype)
 * bf16 working copy s = arena + wb_off + s * P_padded * 2   (only with working_dtype == BF16)
 * stage buffer (e, s) = arena + w_off + (S*(1+e) + s) * P_padded * 4   (only with peer_stage == 1)   */
int hadpsgd_layout(int S, int G, const int64_t* seg_len, int n_seg, hadpsgd_dtypes dt,
                   int64_t* seg_offset, int64_t* P_padded,
                   size_t* w_off, size_t* v_off, size_t* g_off, size_t* wb_off);

/* a1 pairing scheduler (pure host function) -------------------------------------------------- */

/* partner_out[s] = ring neighbour averaged with at step_k.  S==1 -> {0}.  S odd >1 -> INVALID_ARG. */
int hadpsgd_pairing(int S, uint64_t step_k, int32_t* partner_out /*host [S]*/);

/* Parameter-range sharding: rank's contiguous element range [lo, hi) of a
 * P_padded-element buffer split over `world` ranks in whole HADPSGD_SEG_ALIGN_ELEMS blocks
 * (ranges are disjoint, ordered by rank, and cover [0, P_padded); the first P%world ranks get
 * one block more).  P_padded must be a multiple of HADPSGD_SEG_ALIGN_ELEMS (hadpsgd_layout).
 * Pure host function; lo/hi are host out-pointers.                                            */
int hadpsgd_shard_range(int64_t P_padded, int world, int rank, int64_t* lo, int64_t* hi);

/* Learning-rate recipe of PAPER.md:70 (section 3), a host helper that feeds `lr` of
 * hadpsgd_step (row f3): peak = base_lr * total_batch / base_batch (linear scaling); epochs are
 * 1-based; epoch 1 runs at base_lr and the rate rises linearly to peak at epoch warmup_epochs
 * (the paper's example: 0.1 -> 1.0 over 10 epochs for batch 256 -> 2560); afterwards it is
 * annealed by 1/sqrt(2) per epoch.  lr_out: host.  INVALID_ARG on non-positive arguments.     */
int hadpsgd_lr_schedule(double base_lr, double base_batch, double total_batch,
                        int warmup_epochs, int epoch, double* lr_out);

/* lifecycle ---------------------------------------------------------------------------------- */

/* n_seg == 1 is the flat buffer.  opts may be NULL (library-owned memory, default stream,
 * flags 0, current device).  Weights, momenta, gradients and padding start at zero.          */
int hadpsgd_create(int S, int G, const int64_t* seg_len, int n_seg, hadpsgd_dtypes dt,
                   const hadpsgd_opts* opts, hadpsgd_handle* out);
int hadpsgd_destroy(hadpsgd_handle h);

/* a2-a6 the step ----------------------------------------------------------------------------- */

/* Enqueue one fused step on the handle's stream; asynchronous.  Launches per step: ONE for the ring
 * matching or any matching whose members are all paired or all unmixed (up to 32 pairs -- S <= 64 -- per
 * launch); two for a matching that has both (pairs, then singles); on a HADPSGD_PEER handle up to four
 * (pairs / singles, each split into members that first resolve a pending mix and members that do not),
 * back to back with nothing in between.  hadpsgd_launch_count() counts them.
 * S odd and > 1 admits no perfect ring matching (R8): INVALID_ARG unless the handle
 * was created with HADPSGD_NO_MIX -- use hadpsgd_step_matching with an unpaired member instead.
 * Gradient buffers are read-only to the step (not zeroed); w and v are updated in place.
 * step_k is used only for its parity (no hidden counter: a step can be replayed).
 * Launch: the kernel is launched with programmatic stream serialization and waits on the device
 * (griddepcontrol.wait) for the operation before it on the stream, so the usual stream order holds
 * towards every other kernel, copy or event; only capturable into a CUDA graph with a driver that
 * knows programmatic dependencies (CUDA >= 12.3).  The direction of the kernel's walk over the
 * buffers alternates from step to step (L2 reuse): w and v do not depend on it,
 * the diagnostics only in the order their double-precision partial sums are added.             */
int hadpsgd_step(hadpsgd_handle h, float lr, float momentum, uint64_t step_k);

/* Same step, but with a caller-supplied matching (row f1): partner[s] must satisfy
 * partner[partner[s]] == s; partner[s] == s leaves s unmixed (T_ss = 1).  A matching that has
 * both paired and unpaired members is two launches (pairs, then singles), otherwise one.     */
int hadpsgd_step_matching(hadpsgd_handle h, float lr, float momentum, uint64_t step_k,
                          const int32_t* partner /*host [S]*/);

/* End-to-end step from HOST gradients: copies host_grads[s*G+g] (host, P_padded elements of
 * grad_dtype each, ideally pinned) to the device chunk by chunk, overlapping the copies with
 * the fused kernel on element sub-ranges, then copies the diagnostics back into *diag_out
 * (may be NULL) and synchronises the stream.                                                */
int hadpsgd_step_host(hadpsgd_handle h, const void* const* host_grads /*host [S*G]*/,
                      float lr, float momentum, uint64_t step_k, hadpsgd_diag* diag_out);

/* accessors (borrowed device pointers; no copy, no sync) -------------------------------------
 * Without HADPSGD_SHARE_PAIR_WEIGHTS every pointer is fixed for the life of the handle.  With it,
 * hadpsgd_weights / hadpsgd_weights_bf16 return the buffer that holds w_s NOW: it is valid until
 * the next hadpsgd_step* call, pair members return the same pointer, and weights must only be
 * written through it before the first step or after hadpsgd_unshare().                        */
int hadpsgd_weights(hadpsgd_handle h, int s, float** dev_ptr);
/* Gives every super-learner a weight buffer of its own again (copies the shared ones on the
 * stream; asynchronous).  A no-op without HADPSGD_SHARE_PAIR_WEIGHTS or before the first step. */
int hadpsgd_unshare(hadpsgd_handle h);
/* The slot assignment of one step as a pure host function (what hadpsgd_step* does internally):
 * partner [S] is a matching; w_slot [S] in/out = buffer index holding w_s before / after the step;
 * read_slot [S] / write_slot [S] = buffer each member's weights are read from / written to;
 * copy_src / copy_dst [S] receive the *n_copies un-sharing copies that must run first (only when
 * the matching has unmixed members).  share = 0 gives the identity everywhere.                 */
int hadpsgd_plan_slots(int S, const int32_t* partner, int share, int32_t* w_slot, int32_t* read_slot,
                       int32_t* write_slot, int32_t* copy_src, int32_t* copy_dst, int32_t* n_copies);
int hadpsgd_momentum(hadpsgd_handle h, int s, float** dev_ptr);
int hadpsgd_grads(hadpsgd_handle h, int s, int g, void** dev_ptr);
/* bf16 working copy of super-learner s's weights (P_padded bf16 values, rewritten by every step;
 * zero until the first step).  INVALID_ARG unless created with working_dtype == HADPSGD_BF16. */
int hadpsgd_weights_bf16(hadpsgd_handle h, int s, void** dev_ptr);
int hadpsgd_segment(hadpsgd_handle h, int seg, int64_t* elem_offset, int64_t* elem_len);
int hadpsgd_padded_len(hadpsgd_handle h, int64_t* P_padded);

/* Synchronises the stream and copies the diagnostics of the most recent step THAT COMPUTED THEM to the
 * host (host_out->step_k says which).
 * Sharing the device: the cross-block sum of a5 is finished by the LAST blocks of the step's grid, which
 * wait (bounded spin, no fence, no atomics) for partial sums of blocks with lower ids.  On an idle device
 * the whole grid is resident and nothing waits for long.  When the SMs are shared -- several handles on
 * several streams, two processes on one GPU, another library's persistent kernel -- progress relies on
 * the GPU starting the blocks of a grid in block-id order (true of every NVIDIA GPU to date, not a CUDA
 * guarantee); supported and tested: up to 4 handles stepping concurrently on their own streams.  If a
 * collector ever gives up (about a minute), the diagnostics of that step are NaN, the step's w and v are
 * unaffected, and the next hadpsgd_diagnostics() returns HADPSGD_DIAG_TIMEOUT once instead of data.   */
int hadpsgd_diagnostics(hadpsgd_handle h, hadpsgd_diag* host_out);
/* Switch a5 off / on for the steps that follow (default: on, unless created with HADPSGD_NO_DIAG, which
 * cannot be switched on).  A caller that looks at the diagnostics every N steps only pays for them
 * there: for a small problem their final cross-block reduction is most of a step.
 * Results (w, v) do not depend on it.  Host-only state: no stream work.
 * HADPSGD_PEER: pend_wsq / pend_gap of a pending mix are delivered by the launch that RESOLVES it (the
 * next step or hadpsgd_peer_flush); if diagnostics are off for that launch they are never delivered --
 * keep them on for the step after one whose pend_* you want.                                          */
int hadpsgd_set_diagnostics(hadpsgd_handle h, int enable);

/* Consensus distance D = sum_i sum_s (w_s[i] - mean_s w_.[i])^2 of the current weights
 * (mixing alone drives every learner to the mean; D measures how far they are).
 * Optional, NOT part of the step: one extra kernel that reads the S weight buffers once, then
 * synchronises the stream.  D_out: host.  Identity: D(u) - D(w') = 1/2 sum_pairs gap.         */
int hadpsgd_consensus(hadpsgd_handle h, double* D_out);

/* Consensus distance WITHOUT any allocation -- for callers that cannot give this library device memory.
 * hadpsgd_consensus() above needs a handle, and a handle needs an arena (library-cudaMalloc'ed or carved
 * out by the caller).  That is not always possible where D is wanted: the process's framework allocator
 * may already hold nearly all of the GPU (a raw cudaMalloc then fails although the framework has room);
 * a monitor between two steps of a latency-bound loop must not call cudaMalloc / cudaFree, which stall
 * every stream of the device; a hook may only borrow S weight tensors and own no arena at all.  This
 * entry point serves them: it takes the S weight buffers as plain device pointers and writes D to a
 * device double, and its only scratch (one partial sum per thread block + a counter) is a fixed array
 * inside the library image -- HADPSGD_NOALLOC_SCRATCH_BYTES on every GPU that loads the library, held
 * until the process exits.  It calls no cudaMalloc, cudaFree or other allocating routine, on the device
 * or on the host.
 *   w       host array [S] of DEVICE pointers, each to n floats, 16-byte aligned, readable from the
 *           CURRENT device (the call runs on the current device; it does not switch devices)
 *   n       elements per buffer, 0 <= n <= HADPSGD_NOALLOC_MAX_ELEMS; need not be a multiple of 4
 *   D_out   DEVICE pointer to one double (8-byte aligned); written by the kernel, in stream order
 *   stream  cudaStream_t (NULL = legacy default stream); the call only enqueues and returns
 * Same arithmetic as hadpsgd_consensus (mean and deviations in double, fixed summation order): for the
 * same buffers the two agree to the last bit whenever the grids agree (#SMs x 8 <= MAX_BLOCKS blocks).
 * Limits: S > HADPSGD_NOALLOC_MAX_S or n > HADPSGD_NOALLOC_MAX_ELEMS is INVALID_ARG, as are NULL,
 * misaligned or plain-host pointers; the scratch bounds the GRID (HADPSGD_NOALLOC_MAX_BLOCKS), so no n
 * within the limit is refused for lack of scratch.  Text of the last failure on the calling thread:
 * hadpsgd_consensus_noalloc_error().
 *   First call on a device: looks up the device address of the scratch array (cudaGetSymbolAddress) and
 * clears its counter on `stream`; make that call outside any stream capture.  Later calls do neither.
 *   Sharing: every call on a device uses the SAME scratch.  Calls are safe back to back on one stream
 * (or otherwise ordered); two calls whose kernels may overlap on the GPU (different streams, threads or
 * graphs without a dependency) race on it and give garbage -- serialise them.  Each call leaves the
 * counter at zero and overwrites the partials it reads, so nothing has to be cleared in between.      */
#define HADPSGD_NOALLOC_MAX_S 64
#define HADPSGD_NOALLOC_MAX_BLOCKS 2048
#define HADPSGD_NOALLOC_SCRATCH_BYTES ((HADPSGD_NOALLOC_MAX_BLOCKS + 32) * 8) /* 16,640 B per GPU */
#define HADPSGD_NOALLOC_MAX_ELEMS ((int64_t)1 << 36)
int hadpsgd_consensus_noalloc(const float* const* w /*host [S] of dev*/, int S, int64_t n,
                              double* D_out /*dev*/, void* stream);
const char* hadpsgd_consensus_noalloc_error(void);

/* super-learner partition (row f4; Fig. 3) -------------------------------------
 * The paper's topology: every node holds ONE super-learner group and exchanges weights with its ring
 * neighbours.  Here `world` handles ("ranks": one per GPU and process, or several on one device),
 * each created with HADPSGD_PEER and dtypes.peer_stage = 1 over the same segment table, together hold
 * S_global super-learners: rank r owns the global indices [rank_begin[r], rank_begin[r+1]) and S of
 * its hadpsgd_create() call must equal that count.  hadpsgd_step() then uses the ring matching on
 * S_global, and hadpsgd_step_matching() takes partner[S_global].
 *   A pair whose members both live in this handle is mixed as usual.  A member whose partner lives in
 * another handle writes its u = w - lr v' into a STAGE buffer instead (stage parity = epoch & 1) and
 * its mix stays PENDING; the next launch of BOTH owners forms w = 1/2 (u_own + u_partner) on the fly,
 * reading the partner's stage buffer through a peer pointer inside the same fused pass -- 4 B per
 * parameter per pending member cross the link per step, and no kernel ever waits on another one.
 * Same arithmetic as the single-arena step: bit-exact in DETERMINISTIC mode.
 *   Contract: (1) every rank makes the same sequence of step calls with the same matchings (like a
 * collective); each call advances the handle's epoch; (2) hadpsgd_weights(h, s) is INVALID_ARG while s
 * is pending -- call hadpsgd_peer_flush() to materialise every pending mix into the main weight buffers.
 *   Ordering between ranks is the LIBRARY's business (there is no epoch barrier for the caller to
 * provide, and no global one anywhere -- PAPER.md:62 "averages its weights with its neighbor", :66 "removes
 * the global barrier"): every handle owns a 32-bit epoch word behind its stage buffers, writes e + 1 there
 * with a stream memory operation after the last launch of its step e, and before the first launch of a
 * step (or flush) makes its stream wait on the words of exactly the ranks whose stage buffers it is about
 * to read, or which must first have read what it is about to overwrite -- its partners of the last two
 * steps, two ranks in the ring.  The waits are stream operations (cuStreamWaitValue32): no kernel spins
 * and no SM is held, so ranks may share one GPU, run on streams of their own, or live in different
 * processes; a rank that runs ahead simply blocks in its stream until its neighbour has caught up.
 * Consequences: handles that share ONE stream must be stepped epoch by epoch (all handles' step e before
 * any handle's step e + 1 -- the other order waits for a write queued behind itself); a step sequence
 * captured into a CUDA graph replays fixed epoch values and is therefore not ordered by the handshake.
 * hadpsgd_peer_init synchronises the stream once (the word must be zero before peers learn of it).    */

/* rank_begin: host [world+1], increasing, rank_begin[0] = 0, rank_begin[world] = S_global <= HADPSGD_MAX_S. */
int hadpsgd_peer_init(hadpsgd_handle h, int rank, int world, const int32_t* rank_begin);
/* This handle's stage region: dev pointer to [2][S][P_padded] floats (stage parity, local member). */
int hadpsgd_peer_stage(hadpsgd_handle h, float** dev_ptr);
/* Tell this handle where rank r's stage region is: a dev pointer VALID IN THIS PROCESS AND ON THIS
 * DEVICE'S KERNELS (the same device, or a peer device with access enabled by the caller).  Every
 * rank other than the handle's own must be attached before the first step.                       */
int hadpsgd_peer_attach(hadpsgd_handle h, int r, const float* stage_region_of_rank_r);
/* Across processes: export this handle's arena as a CUDA IPC handle (ipc_handle_out: host, 64 bytes)
 * plus the byte offset of the stage region from the exported allocation's base ...
 * A CUDA IPC handle names a whole ALLOCATION, so the importing process can read everything that
 * shares the arena's cudaMalloc block.  Create handles that will be exported with opts->arena = NULL
 * (library-owned: the allocation is exactly the arena) or over a dedicated cudaMalloc of your own.  A
 * slice of a framework's caching allocator exposes that allocator's whole segment to the peer -- unrelated
 * tensors included -- and memory from cudaMallocAsync pools or virtual-memory ("expandable") segments
 * cannot be exported this way at all (cudaIpcGetMemHandle fails: HADPSGD_CUDA).                      */
int hadpsgd_peer_ipc_export(hadpsgd_handle h, void* ipc_handle_out, uint64_t* stage_offset_out);
/* ... and open rank r's export in this process (cudaIpcOpenMemHandle with lazy peer access), then
 * attach it.  One mapping per rank: attaching rank r again synchronises the stream, closes r's
 * previous mapping and opens the new one; hadpsgd_destroy() closes what is left.                    */
int hadpsgd_peer_ipc_attach(hadpsgd_handle h, int r, const void* ipc_handle, uint64_t stage_offset);
/* Materialise every pending mix: w_s = 1/2 (u_own + u_partner) into the main weight buffer (one small
 * kernel on the stream; asynchronous), delivering pend_wsq / pend_gap.  It first waits, on the stream,
 * for the partners' publishing step (epoch handshake).  Not a step: the epoch does not advance, ranks
 * need not call it together.  A rank must not destroy its handle (or free its arena) while a partner
 * may still flush or step against it: agree on teardown outside this library.                      */
int hadpsgd_peer_flush(hadpsgd_handle h);
/* The peer plan of one step as a pure host function (no GPU): see csrc/scheduler.cpp.  pending: in/out
 * [S_local] (global partner index or -1); outputs [S_local]: kind (0 pair member, 1 unmixed,
 * 2 straddling), mate (local pair mate or -1), read_buf / write_buf (weight buffer index: main s,
 * stage (e, s) = S_local (1 + e) + s), read_peer (-1 or e * S_global + global partner).           */
int hadpsgd_plan_peer(int world, int rank, const int32_t* rank_begin, const int32_t* partner /*[S_global]*/,
                      uint64_t epoch, int32_t* pending, int32_t* kind, int32_t* mate, int32_t* read_buf,
                      int32_t* write_buf, int32_t* read_peer);

/* Measurement knob: resident blocks per SM of the persistent grid (1..16, clamped to what fits);
 * 0 restores the default chosen per (G, dtype, mode).  w and v do not depend on it; the diagnostics
 * only in the order their partial sums are added (same shape, same bits).                     */
int hadpsgd_set_launch(hadpsgd_handle h, int blocks_per_sm);
/* Number of kernel launches issued by this handle so far (bench.py's gpu_launches). */
int hadpsgd_launch_count(hadpsgd_handle h, uint64_t* out);

/* Thread safety: the pure host functions above are re-entrant.  A handle is NOT thread-safe: calls on
 * one handle must be serialised by the caller; different handles may be used from different threads. */
const char* hadpsgd_error_string(int code);
const char* hadpsgd_last_error(hadpsgd_handle h);

#ifdef __cplusplus
}
#endif
#endif
