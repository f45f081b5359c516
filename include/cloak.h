/* cloak.h -- C ABI of the B200-native CloakLM cloaked-layout hot path (libcloak.so).
 *
 * What this library is.  CloakLM (arxiv/paper_2606_18400) obfuscates where an LLM's weights sit in
 * HBM while the authorised reader keeps an unchanged logical view.  The paper does it with a
 * random permutation computed before any page is allocated or any weight transferred
 * (section 5), a random virtual->physical map of 2 MB pages through the CUDA VMM API
 * (Table 1b :192-201), a random tensor order (Table 1a
 * :181-190) and "inter- and intra-layer weight shuffling".  BASELINE.json's
 * north_star fixes the calls: a keyed Philox4x32-10 permutation, a block scatter into a 2 MiB page
 * pool, a function-preserving neuron/head permutation and a GEMV/GEMM that reads through the
 * block table.  Concrete definitions (counter layout, direction of the table, padding, tile
 * layout) are the readings O1-O12 / G1-G22 of SURVEY.md section 8(c), restated in DESIGN.md.
 *
 * Conventions.
 *   - Every function returns a cloak_status: 0 = CLOAK_OK, negative = error.  No exceptions, no
 *     aborts, no printing.  cloak_last_error() returns a thread-local, library-owned C string
 *     describing the last failure on the calling thread.
 *   - "d_" arguments are DEVICE pointers, "h_" arguments are HOST pointers.  The caller owns every
 *     tensor it passes; the library owns pools and their tables.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Every
 *     device-side call is asynchronous on that stream and never synchronises it, except where
 *     stated (pool create/destroy, *_host convenience calls).
 *   - There is no CPU fallback: without a CUDA device every compute call fails with
 *     CLOAK_ERR_CUDA.
 */
#ifndef CLOAK_H_
#define CLOAK_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    CLOAK_OK = 0,
    CLOAK_ERR_INVALID = -1,     /* null pointer, n == 0, batch out of range, size mismatch          */
    CLOAK_ERR_ALIGN = -2,       /* pointer / offset / size not 16-byte or block aligned             */
    CLOAK_ERR_UNSUPPORTED = -3, /* dtype / layout / block-size combination not implemented          */
    CLOAK_ERR_OOM = -4,         /* device or host allocation failed                                 */
    CLOAK_ERR_CUDA = -5         /* driver / runtime error; text in cloak_last_error()               */
} cloak_status;

typedef enum { CLOAK_F32 = 0, CLOAK_BF16 = 1 } cloak_dtype;

/* Storage layout of a logical [N, K] matrix inside the arena.
 * ROWMAJOR: the tensor's bytes as given.  TILE128: tile (tn, tk) of 128 x 128 elements sits at tile
 * index tn*(K/128)+tk; element (r, c) at element offset r*128+c inside the tile; no swizzle. */
typedef enum { CLOAK_ROWMAJOR = 0, CLOAK_TILE128 = 1 } cloak_layout;

const char* cloak_last_error(void);

/* Library version / build info: a static string such as "cloak-b200 0.1 sm_100a". */
const char* cloak_version(void);

/* Facts the library found out at run time, as a thread-local string for logs and bench lines: whether the driver accepted
 * the cooperative GEMV launch together with programmatic dependent launch, kernels launched so far. */
const char* cloak_runtime_info(void);

/* Process-wide number of CUDA kernels this library has launched so far (for bench.py's gpu_launches). */
uint64_t cloak_launch_count(void);

/* ---- S1 keyed permutation (north_star: "indices sorted by Philox(key, index)").
 * For i in [0, n): o = Philox4x32-10(ctr = (i, 0, stream_id lo, stream_id hi), key = (key lo, key hi)),
 * r_i = o[0]:o[1]; perm = indices sorted ascending by (r_i, i); inv[perm[j]] = j.
 * d_perm / d_inv: caller-owned device buffers of n uint32; either may be NULL (not both).
 * n in [1, 2^28].  Asynchronous on `stream` (workspace comes from the library's own stream-ordered memory pool, which keeps
 * at most 512 MiB of freed scratch cached; the process's default pool is not touched). */
cloak_status cloak_keygen(uint64_t key, uint64_t stream_id, uint32_t n,
                          uint32_t* d_perm, uint32_t* d_inv, void* stream);

/* ---- S2 page pool ("CUDA VMM ... tensor pointers unchanged").
 * Geometry: nb = ceil(payload/block), bpp = page/block, npages = ceil(nb/bpp), nslots = npages*bpp.
 * Tables: (blockperm, blockinv) = keygen(key, 1<<32, nslots); (pageperm, pageinv) = keygen(key, 2<<32, npages).
 * Real pages (page_bytes a multiple of the VMM granularity and PLAIN_ALLOC not set): a VA range of
 * npages*page_bytes is reserved, one physical handle per page is created (creation order stands for
 * physical order, G6), and handle pageinv[v] is mapped at VA page v; the authorised table is
 * T[i] = blockinv[i].  Emulated pages (any other page size, or PLAIN_ALLOC): one allocation that *is*
 * the dump view D; T[i] = pageinv[blockinv[i]/bpp]*bpp + blockinv[i]%bpp.
 * The pool memory is zero-filled.  block_bytes must be a power of two >= 16 and divide page_bytes.
 * Synchronous (driver calls + one stream sync). */
typedef struct cloak_pool cloak_pool;
enum {
    CLOAK_POOL_IDENTITY = 1,     /* identity block + page tables: the "native" layout              */
    CLOAK_POOL_PLAIN_ALLOC = 2   /* one plain allocation instead of per-page VMM handles           */
};
cloak_status cloak_pool_create(int device, uint64_t payload_bytes, uint32_t block_bytes,
                               uint64_t page_bytes, uint64_t key, uint32_t flags, cloak_pool** out);
cloak_status cloak_pool_destroy(cloak_pool* pool);

/* Any output pointer may be NULL.  *d_base: device address of the pool (the VA view V for real pages -- its first half: a pool of
 * real pages reserves twice its size of virtual addresses, and after a cloak_rekey_pages_* a page may live in the second half,
 * nslots*block bytes further on, which the table T accounts for -- the dump view D for emulated pages).  *d_table: device array T[0..nb).  *is_vmm: 1 for real pages. */
cloak_status cloak_pool_info(const cloak_pool* pool, void** d_base, const uint32_t** d_table,
                             uint32_t* nb, uint32_t* nslots, uint32_t* npages, int* is_vmm);

/* Host copies of the four tables (caller-owned host arrays; any may be NULL): blockperm/blockinv have
 * nslots entries, pageperm/pageinv npages.  Synchronous. */
cloak_status cloak_pool_tables(const cloak_pool* pool, uint32_t* h_blockperm, uint32_t* h_blockinv,
                               uint32_t* h_pageperm, uint32_t* h_pageinv);

/* Copies the dump view D (pages in physical = handle-creation order, O5) into d_out (nslots*block bytes).
 * Real pages: read through a second (alias) mapping of the same handles in creation order.
 * Emulated pages: a plain copy of the pool.  Asynchronous on `stream`. */
cloak_status cloak_pool_dump(const cloak_pool* pool, void* d_out, void* stream);

/* Milliseconds the host-side mapper (reserve/create/map/set-access) took in cloak_pool_create. */
cloak_status cloak_pool_map_ms(const cloak_pool* pool, double* ms);
/* ... and its three phases: cuMemCreate of every page, cuMemMap in keyed order, cuMemSetAccess (0 for emulated pools). */
cloak_status cloak_pool_map_phases(const cloak_pool* pool, double* create_ms, double* map_ms, double* access_ms);

/* Layout-quality report (the paper's only security-side metric that needs no attacker is a
 * contiguity percentage).  Fractions of logical neighbours that are still neighbours:
 *   *va_blocks       = #{i : T_va[i+1] == T_va[i] + 1} / (nb - 1),  T_va[i] = blockinv[i]   (the VA view V)
 *   *physical_blocks = the same through the page map, slot(i) = pageinv[blockinv[i] / bpp] * bpp + blockinv[i] % bpp
 *                      (the dump view D: what reading pages in physical order sees; G8: expect about 1 / nslots)
 *   *pages           = #{v : pageinv[v+1] == pageinv[v] + 1} / (npages - 1)
 * An identity pool reports 1, 1, 1.  Any output may be NULL.  Runs on `stream` and synchronises that stream only. */
cloak_status cloak_pool_adjacency(const cloak_pool* pool, double* va_blocks, double* physical_blocks, double* pages,
                                  void* stream);

/* The full report, for the same three sequences: a RUN is a maximal stretch of logically consecutive
 * items (blocks, pages) that are still consecutive in that view -- what an observer reading memory in the view's order can stitch
 * together without the key.  items = nb (blocks) or npages; runs = number of runs (an identity pool: 1); longest_run;
 * items_in_runs_of_2_or_more; adjacent_fraction = (items - runs) / (items - 1) (= cloak_pool_adjacency's number);
 * histogram[k] = runs of length L with 2^k <= L < 2^(k+1).  The paper's metric is "virtual address ranges backed by contiguous
 * physical pages", 91.41 % -> 2.38 % and 95.57 % -> 1.57 % (its unit is undefined, G12): `pages` is the closest
 * analogue.  Computed on the GPU; runs on `stream` and synchronises that stream only. */
typedef struct {
    uint64_t items, runs, longest_run, items_in_runs_of_2_or_more;
    double adjacent_fraction;
    uint64_t histogram[32];
} cloak_run_stats;
typedef struct {
    cloak_run_stats va_blocks, physical_blocks, pages;
} cloak_layout_report;
cloak_status cloak_pool_layout_report(const cloak_pool* pool, cloak_layout_report* h_report, void* stream);

/* ---- S4 block shuffle / unshuffle, S8 re-layout (north_star (a)).
 * shuffle:   pool[T[i]*b + o] = logical[i*b + o] for the arena range [logical_offset, +bytes);
 * unshuffle: logical[i*b + o] = pool[T[i]*b + o] for the same range.
 * d_logical points at the first byte of that range (e.g. a tensor's data), 16-byte aligned.
 * logical_offset must be a block multiple; bytes a 16-byte multiple.  A final partial block is
 * zero-padded on shuffle (G4) and truncated on unshuffle.  Asynchronous on `stream`. */
cloak_status cloak_shuffle(cloak_pool* pool, const void* d_logical, uint64_t logical_offset,
                           uint64_t bytes, void* stream);
cloak_status cloak_unshuffle(const cloak_pool* pool, void* d_logical, uint64_t logical_offset,
                             uint64_t bytes, void* stream);
/* The same for n arena ranges in one launch (per 128 ranges): range r is h_bytes[r] bytes at arena offset h_offsets[r],
 * in the caller's device buffer d_logical[r]; h_logical pointers, offsets and sizes are HOST arrays of n entries, not
 * referenced after the call returns.  Ranges must not overlap.  A model is hundreds of tensors and one launch per tensor
 * leaves the small ones launch-bound.  Asynchronous on `stream`. */
cloak_status cloak_shuffle_many(cloak_pool* pool, uint32_t n, const void* const* d_logical,
                                const uint64_t* h_offsets, const uint64_t* h_bytes, void* stream);
cloak_status cloak_unshuffle_many(const cloak_pool* pool, uint32_t n, void* const* d_logical,
                                  const uint64_t* h_offsets, const uint64_t* h_bytes, void* stream);
/* pool_b[T_b[i]] = pool_a[T_a[i]] for every logical block, without materialising the arena.
 * Both pools must have the same payload and block size.  Asynchronous on `stream`. */
cloak_status cloak_relayout(const cloak_pool* from_a, cloak_pool* to_b, void* stream);

/* Re-key the block permutation of a pool IN PLACE ("reshuffled periodically ...
 * no additional memory footprint"): afterwards the pool holds, under the block tables of `new_key` and its unchanged page
 * map, exactly what it held before:  pool[T_new[i]] = old pool[T_old[i]]  for every block slot i, bit for bit what
 * cloak_relayout into a second pool would give, zero pad slots included.  Pages are not re-mapped.  The only extra memory
 * is a spare buffer of about spare_bytes (0 = one page): the permutation's cycles are cut into segments whose first block
 * is saved there, and the more segments, the more of them move in parallel (one page is enough for full speed only on
 * pools of a few hundred MB; 1/64 of the pool is on any).  The cycle decomposition runs on the host: the call
 * synchronises `stream` and returns when the pool is re-keyed; GEMVs issued afterwards read through the new table. */
cloak_status cloak_rekey_inplace(cloak_pool* pool, uint64_t new_key, uint64_t spare_bytes, void* stream);

/* Re-randomise the PHYSICAL PAGE MAP of a pool under live decode ("At initialization and
 * then periodically randomizes the mapping of virtual addresses to physical HBM pages", :205-207 "using CUDA VMM APIs ... The only
 * overhead arises from synchronization points needed to safely remap pages", cadence :207 / :283).
 * (pageperm', pageinv') = keygen(new_key, 2<<32, npages).  Afterwards VA page v is backed by physical page pageinv'[v] (physical
 * index = handle-creation order, G6): the dump view becomes D'[pageinv'[v]*P + o] = D[pageinv[v]*P + o]; the VA view, the block
 * tables' logical content and every result read through the pool are unchanged, bit for bit.  Real (VMM) pages only.
 *   _begin   draws the new page map (synchronises `stream` once), creates `spare_pages` (1..64; 0 = 1) spare physical pages: the
 *            only extra memory, released when the re-key completes.  One re-key per pool at a time.
 *   _step    NON-BLOCKING, to be called between decode steps: unmaps the old addresses of the moves the stream has passed, and
 *            starts up to max_moves (<= 16) new page moves -- cuMemMap of the destination physical page at the page's address in the
 *            OTHER half of the pool's (doubled) virtual range, then on `stream` a 2 MiB copy and the switch of the page's block-table
 *            entries.  Kernels launched before the switch read the old address, kernels launched after it the new one; CUDA graphs
 *            of cloak_gemv_chain / cloak_gemm_chain stay valid (they hold the table's address, not its contents).  With k spare
 *            pages k cycles of the page permutation are followed at once, one move each per call.  *h_remaining (may be NULL) =
 *            pages not yet home; 0 means the re-key is complete and cloak_pool_tables / cloak_pool_dump show the new map.
 *            Host cost: ~0.3 ms of driver calls per move on B200, on the calling thread, while the GPU runs what was launched before.
 *   _finish  runs the remaining moves to the end, waiting for each batch (the stop-the-world form), and synchronises `stream`.
 * While a re-key is in progress, all calls on the pool must be issued on that one `stream`; cloak_rekey_inplace is refused;
 * cloak_pool_info's d_base addresses half 0 only (tests read the VA view through cloak_unshuffle). */
cloak_status cloak_rekey_pages_begin(cloak_pool* pool, uint64_t new_key, uint32_t spare_pages, void* stream);
cloak_status cloak_rekey_pages_step(cloak_pool* pool, uint32_t max_moves, void* stream, uint32_t* h_remaining);
cloak_status cloak_rekey_pages_finish(cloak_pool* pool, void* stream);

/* Host-buffer variants (end-to-end path): h_logical is a HOST buffer (pinned for full speed); the
 * library stages it through device memory in chunks.  They synchronise `stream` before returning. */
cloak_status cloak_shuffle_host(cloak_pool* pool, const void* h_logical, uint64_t logical_offset,
                                uint64_t bytes, void* stream);
cloak_status cloak_unshuffle_host(const cloak_pool* pool, void* h_logical, uint64_t logical_offset,
                                  uint64_t bytes, void* stream);

/* Selects the copy engine used by shuffle / unshuffle / relayout: 0 = automatic, 1 = 16-byte
 * LDG/STG, 2 = TMA bulk copy through a shared-memory ring.  For A/B measurement; process-wide. */
cloak_status cloak_set_copy_engine(int engine);

/* L2 eviction hints of the TMA copy engine: bit 0 = its stores are evict_first, bit 1 = its loads are.  Meant to keep a streaming
 * copy from leaving the 126 MB L2 full of dirty lines that the next kernel then pays to write back (the GEMV that follows a
 * re-layout runs 90 us instead of 80); measured on B200: the hint changes neither the copy nor its successor, so the default is 0
 * (none).  For A/B measurement; process-wide. */
cloak_status cloak_set_copy_cache_hint(int hint);

/* ---- S3 tensor order.  Host helper, no device work.
 * (order, _) = keygen(key, 3<<32, T); the arena holds tensors order[0], order[1], ... back to back, each
 * padded to a multiple of block_bytes.  h_offsets_out: T entries; h_total_out: padded arena bytes. */
cloak_status cloak_arena_plan(uint64_t key, uint32_t T, const uint64_t* h_bytes, uint32_t block_bytes,
                              uint64_t* h_offsets_out, uint64_t* h_total_out);

/* ---- S5 neuron / head permutation (north_star (b)).  Out of place; src and dst of one
 * tensor have the same shape and must not overlap; any src/dst pair may be NULL/NULL to skip it.
 * Shapes (row-major, [out, in]): gate, up [inter, hidden]; down [hidden, inter]; q [n_q*head_dim, hidden];
 * k, v [n_kv*head_dim, hidden]; o [hidden, n_q*head_dim].
 *   (pi, _) = keygen(key, (4<<32)|layer, inter): gate'[r,:] = gate[pi[r],:], up' likewise, down'[:,r] = down[:,pi[r]]
 *   (kappa, _) = keygen(key, (5<<32)|layer, n_kv); (rho_g, _) = keygen(key, (6<<32)|(layer*n_kv+g), n_q/n_kv);
 *   eta[g*G+j] = kappa[g]*G + rho_g[j]; k', v' row groups by kappa; q' row groups and o' column groups by eta.
 * Asynchronous on `stream`. */
typedef struct {
    uint32_t hidden, inter, n_q, n_kv, head_dim;
    cloak_dtype dt;
    uint32_t layer;
} cloak_block_shape;
cloak_status cloak_permute_mlp_heads(uint64_t key, const cloak_block_shape* shape,
                                     const void* d_gate, const void* d_up, const void* d_down,
                                     const void* d_q, const void* d_k, const void* d_v, const void* d_o,
                                     void* d_gate_o, void* d_up_o, void* d_down_o,
                                     void* d_q_o, void* d_k_o, void* d_v_o, void* d_o_o, void* stream);

/* Column gather of 2-byte elements (down's columns): 0 = automatic (two source rows interleaved into 32-bit pairs in shared
 * memory, one LDS per output element PAIR), 1 = the element-by-element gather.  For A/B measurement; process-wide. */
cloak_status cloak_set_gather_engine(int engine);

/* ---- S5 for mixture-of-experts layers (the paper evaluates Qwen3-MoE).
 * Shapes (row-major, contiguous): router [n_experts, hidden]; gate, up [n_experts, inter, hidden]; down [n_experts, hidden, inter].
 *   (eps, _)  = keygen(key, (7<<32)|layer, n_experts):  new expert e' is old expert eps[e'];  router'[e',:] = router[eps[e'],:]
 *   (pi_e, _) = keygen(key, (8<<32)|(layer*n_experts + e), inter) for every OLD expert e, and with e = eps[e']:
 *               gate'[e'] = gate[e][pi_e,:],  up'[e'] = up[e][pi_e,:],  down'[e'] = down[e][:,pi_e]
 * The sparse MLP (top-k by router logit, softmax over the selected logits) is unchanged as a function.  Out of place, all
 * four tensors required.  Asynchronous on `stream`.  bf16 experts with inter <= 4096 (rows of `down` up to 8 KiB) take five
 * launches per layer -- one keygen launch for all experts' pi, one row gather each over the stacked gate and up, one column
 * gather over all `down` matrices (Qwen3-MoE-shaped layer, 2.4 GB moved: 0.48 ms = 5.0 TB/s); other shapes and f32 go expert
 * by expert, a few launches each. */
typedef struct {
    uint32_t hidden, inter, n_experts;
    cloak_dtype dt;
    uint32_t layer;
} cloak_moe_shape;
cloak_status cloak_permute_experts(uint64_t key, const cloak_moe_shape* shape, const void* d_router, const void* d_gate,
                                   const void* d_up, const void* d_down, void* d_router_o, void* d_gate_o, void* d_up_o,
                                   void* d_down_o, void* stream);

/* ---- S5 + S4 in one pass: the fused load path (the layout is decided before
 * any weight lands).  Same permutation as cloak_permute_mlp_heads, but every permuted tensor is written straight into
 * `pool` through its block table at arena byte offset h_offsets[i] (i = gate, up, down, q, k, v, o; a block
 * multiple; ignored where the source is NULL), CLOAK_ROWMAJOR.  The pool bytes afterwards equal those of
 * cloak_permute_mlp_heads followed by cloak_shuffle of each tensor (the tail of a final partial block is zeroed),
 * at 2 bytes of traffic per payload byte instead of 4.  h_offsets is a HOST array of 7.  Asynchronous on `stream`. */
cloak_status cloak_load_mlp_heads(uint64_t key, const cloak_block_shape* shape, cloak_pool* pool,
                                  const void* d_gate, const void* d_up, const void* d_down,
                                  const void* d_q, const void* d_k, const void* d_v, const void* d_o,
                                  const uint64_t* h_offsets, void* stream);

/* ---- S3 + S5 + layout + S4 in one pass: the load path of a whole model (PAPER.md:173-177 the load is
 * "the only phase in which the full set of weight transfers crosses the PCIe bus", Tier 1 hides its order; :217 the permutation
 * and the pages are decided before any weight is transferred).
 * Each item is one tensor of a decoder layer (role GATE .. O: shape from `shape`, permutation that of cloak_permute_mlp_heads
 * for item.layer -- shape->layer is ignored) or a PLAIN [N, K] matrix that is not permuted (embeddings, lm_head, a router).
 * The tensor is read ONCE from item.src -- a device pointer, or a pointer to pinned (page-locked, device-mapped) host memory,
 * which the gather kernels then read across PCIe themselves: no staging copy (pageable host memory is refused with
 * CLOAK_ERR_INVALID) -- and written straight through the pool's block
 * table at arena byte item.arena_offset (a block multiple) in `layout` (CLOAK_ROWMAJOR, or CLOAK_TILE128: the storage
 * conversion is an address computation in the same pass; N and K multiples of 128).  The pool bytes afterwards equal those of
 * cloak_permute_mlp_heads (-> cloak_to_tile128) -> cloak_shuffle, tail of a final partial block zeroed: 2 bytes of traffic per
 * payload byte instead of 4 or 6.  The items are issued in ascending arena_offset, i.e. in cloak_arena_plan's keyed tensor
 * order, whatever order the caller lists them in.  h_items is a HOST array, not referenced after the call returns; ranges must
 * not overlap.  Asynchronous on `stream`. */
typedef enum { CLOAK_ROLE_GATE = 0, CLOAK_ROLE_UP = 1, CLOAK_ROLE_DOWN = 2, CLOAK_ROLE_Q = 3, CLOAK_ROLE_K = 4,
               CLOAK_ROLE_V = 5, CLOAK_ROLE_O = 6, CLOAK_ROLE_PLAIN = 7 } cloak_role;
typedef struct {
    const void* src;
    uint64_t arena_offset;
    uint32_t layer;
    uint32_t role;      /* cloak_role */
    uint32_t N, K;      /* CLOAK_ROLE_PLAIN only */
} cloak_load_item;
cloak_status cloak_load_tensors(uint64_t key, const cloak_block_shape* shape, cloak_pool* pool,
                                const cloak_load_item* h_items, uint32_t n, cloak_layout layout, void* stream);

/* Storage-layout conversion ROWMAJOR -> TILE128 of a logical [N, K] matrix (N, K multiples of 128).
 * Out of place.  Asynchronous on `stream`. */
cloak_status cloak_to_tile128(const void* d_src, void* d_dst, uint32_t N, uint32_t K, cloak_dtype dt,
                              void* stream);

/* ---- S6 / S7 the authorised read (north_star (c)).
 * Y[m, n] = sum_k X[m, k] * W[n, k].  W lives in the pool at arena byte offset w_offset (a block
 * multiple), logical shape [N, K], read through the pool's table T.  X [batch, K] and Y [batch, N] are
 * row-major device buffers of W's dtype, 16-byte aligned.  Accumulation is fp32.
 * cloak_gemv: batch 1..16, layout ROWMAJOR, K a multiple of 64 and N of 16 (bf16) / K of 4 (f32).
 *             Stream order: X, Y and the library's scratch are touched in stream order.  The bf16 streaming
 *             kernel is launched with programmatic dependent launch and may begin fetching W while the
 *             preceding kernel of `stream` drains; the library withholds that for the first GEMV that follows
 *             a cloak_shuffle* / cloak_relayout into the pool (those calls mark the pool).  Code that writes
 *             pool memory by other means (through cloak_pool_info's d_base) must synchronise before the
 *             next cloak_gemv.
 * cloak_gemm: batch 1..256 (the MMA runs on the batch rounded up to a multiple of 16; the extra X rows are zero-filled by
 * TMA and their outputs are not stored), dtype BF16, layout TILE128, block_bytes >= 32 KiB
 *             (tcgen05 tensor cores, accumulators in TMEM, tiles fetched by TMA through the table).
 * Asynchronous on `stream`; no compute call synchronises or calls the driver's allocator.
 * Scratch (split-K counters and fp32 partials) belongs to the pool.  16 MiB exist from cloak_pool_create on: enough for every
 * cloak_gemv / cloak_gemv_chain of the streaming kernel and for small GEMMs.  A call that needs more (the cloak_*_scratch_bytes
 * queries below say how much) grows the scratch in the order of ITS stream (stream-ordered allocation, counters zeroed on
 * that stream, the old buffer released behind the kernels already queued) -- except while that stream is being captured into
 * a CUDA graph, where the call fails with CLOAK_ERR_INVALID: reserve first.  With the scratch reserved, a first-use call can
 * be captured without any warm-up.  The counters and partials are shared by all calls on one pool: those calls must be
 * ordered with respect to each other (one stream, or events), and replays of one graph must not overlap each other.
 * Different pools are independent and may run on different streams at the same time.
 * Co-residency.  A cloak_gemv_chain launch that contains an `after` op has a grid-wide barrier inside and is launched as a
 * COOPERATIVE grid (all CTAs resident, or the launch waits / fails -- never a hang when other kernels hold SMs, e.g. two pools'
 * chains on two streams).  In launches without one (cloak_gemv, chains of independent ops) a CTA -- its helper warp, not the warps
 * that stream -- waits only for the partials of the few CTAs that hold the NEXT ranges of the same op.  Those stay ordinary
 * launches: they need the whole grid (one CTA per SM, never more CTAs than the device has SMs) to become resident, which the
 * GPU's in-order dispatch of grids gives whenever all SMs of the device are available to the context, whatever else is queued.
 * A context confined to FEWER SMs than the device reports (MPS active-thread percentage, green contexts) cannot hold the grid:
 * use cloak_set_gemv_engine(1) there (the one-shot kernel waits for nobody).  The GEMM waits
 * only for partials of CTAs that drew their ticket before the waiter, i.e. that are already running: no assumption at all. */
typedef struct {
    uint64_t w_offset;
    uint32_t N, K;
    cloak_dtype dt;
    cloak_layout layout;
} cloak_tensor;
cloak_status cloak_gemv(const cloak_pool* pool, const cloak_tensor* w, const void* d_x, void* d_y,
                        uint32_t batch, void* stream);
cloak_status cloak_gemm(const cloak_pool* pool, const cloak_tensor* w, const void* d_x, void* d_y,
                        uint32_t batch, void* stream);
/* cloak_gemv without any allocation (north_star (c): the same cloaked GEMV; for callers that cannot call
 * cudaMalloc -- code under CUDA graph capture, tight serving loops, harnesses that forbid it).  Same contraction, same kernel
 * and same results as cloak_gemv's streaming path, bit for bit; the kernel's scratch (row-tile arrival counters and the fp32
 * partials of row tiles cut by a range boundary) lives in a fixed 512 KiB `static __device__` array of the library instead of
 * the pool's workspace, so the call never calls cudaMalloc / cudaFree / cudaMallocAsync or any allocating routine, whatever
 * the pool's workspace state.  Every GPU that loads the library holds those 512 KiB until the process exits.
 * Limits: CLOAK_BF16, CLOAK_ROWMAJOR, K % 256 == 0, N % 16 == 0, block_bytes >= 512, batch 1..16 (else CLOAK_ERR_UNSUPPORTED /
 * CLOAK_ERR_INVALID), and N <= 524 288 rows (one counter per 8 rows; beyond that CLOAK_ERR_UNSUPPORTED, nothing launched:
 * use cloak_gemv).  d_x [batch, K] and d_y [batch, N] are DEVICE buffers of the caller, as in cloak_gemv.
 * ALL calls, on every pool and stream of a device, share the one array, and it keeps the last call's contents: each call
 * first clears the counters it uses (a small kernel on `stream`) and writes its partials before it reads them, so calls in
 * stream order are independent of what ran before; two calls that OVERLAP on the GPU (different streams with no event between
 * them, concurrent graph branches) race on the array and give wrong results.  Asynchronous on `stream`; two launches. */
cloak_status cloak_gemv_static(const cloak_pool* pool, const cloak_tensor* w, const void* d_x, void* d_y,
                               uint32_t batch, void* stream);
/* Bytes of pool scratch the chain calls below need for these ops at this batch (the largest of the launches they split into);
 * host only.  cloak_pool_reserve_workspace grows the pool's scratch to at least `bytes` (never shrinks); synchronous: it
 * waits for the device, so call it at load time.  (cloak_gemv / cloak_gemm = a chain of one op.) */
struct cloak_gemv_op;
struct cloak_gemm_op;
cloak_status cloak_gemv_chain_scratch_bytes(const cloak_pool* pool, const struct cloak_gemv_op* h_ops, uint32_t n_ops,
                                            uint32_t batch, uint64_t* h_bytes);
cloak_status cloak_gemm_chain_scratch_bytes(const cloak_pool* pool, const struct cloak_gemm_op* h_ops, uint32_t n_ops,
                                            uint32_t batch, uint64_t* h_bytes);
cloak_status cloak_pool_reserve_workspace(cloak_pool* pool, uint64_t bytes);

/* A chain of GEMVs over one pool in ONE persistent launch (SURVEY.md 8(a) S6 at cfg2: "end-to-end cloaked decode
 * of all layers' projection GEMVs"; decode is bandwidth-bound, so the weight stream should
 * never stop).  Op i computes Y_i = X_i W_i^T like cloak_gemv, with two additions:
 *   - d_gate / d_act, both or neither: the op ALSO writes d_act[m, n] = silu(d_gate[m, n]) * Y_i[m, n] ([batch, N],
 *     fp32 arithmetic on the bf16 values, rounded to bf16 exactly as cloak_silu_mul does; O9: the gated MLP's
 *     activation, fused into the up projection's epilogue).  d_gate must be the d_y of an earlier op of this
 *     chain with the same N and K (the usual gate projection), or a buffer complete before the call;
 *   - after != 0 says that X_i is written by an earlier op of this chain.  after == 1: the op starts only when ALL
 *     earlier ops have completed (one grid-wide arrival).  after == 2: it has the same dependency as the nearest
 *     earlier op with after != 0 and shares that arrival -- e.g. the down projections of several experts, all of which
 *     follow all the up projections: the first says 1, the others 2.  (In a split chain -- more than 48 ops, or mixed
 *     chunk sizes -- after == 2 on the first op of a launch needs nothing: the launch boundary orders it.)
 *     Ops with after == 0 must not read what earlier ops of the chain write.
 * The weight stream of op i+1 is already being fetched while op i finishes, dependent or not.
 * All ops: CLOAK_BF16, CLOAK_ROWMAJOR, K % 256 == 0, N % 16 == 0, pool block_bytes >= 512, batch 1..16, outputs
 * distinct.  h_ops is a HOST array (copied into the launch parameters; not referenced after the call returns).
 * Chains longer than 48 ops, or mixing row sizes that need different chunk sizes, are split into several
 * launches (stream order keeps the semantics).  Asynchronous on `stream`. */
typedef struct cloak_gemv_op {
    cloak_tensor w;
    const void* d_x;
    void* d_y;
    const void* d_gate;
    void* d_act;
    uint32_t after;
} cloak_gemv_op;
cloak_status cloak_gemv_chain(const cloak_pool* pool, const cloak_gemv_op* h_ops, uint32_t n_ops, uint32_t batch,
                              void* stream);
/* A list of INDEPENDENT GEMMs over one pool in one persistent launch (per 16 ops): Y_i = X_i W_i^T as in cloak_gemm;
 * every op has its own output and no op may read what another op of the list writes.  The tiles of all ops of a launch
 * form ONE sequence that is cut into chunks (cloak_set_gemm_schedule): K is split where those boundaries fall, so a
 * chain is deterministic and the same on cloaked and identity-table pools, and equals cloak_gemm up to the fp32
 * summation order.  The weight stream runs on across op boundaries
 * (BASELINE.json configs[3]: "cloaked decode GEMM" of every projection of the model).  h_ops is a HOST array, not
 * referenced after the call returns.  Asynchronous on `stream`. */
typedef struct cloak_gemm_op {
    cloak_tensor w;
    const void* d_x;
    void* d_y;
} cloak_gemm_op;
cloak_status cloak_gemm_chain(const cloak_pool* pool, const cloak_gemm_op* h_ops, uint32_t n_ops, uint32_t batch,
                              void* stream);
/* Selects the bf16 GEMV kernel: 0 = automatic (streaming TMA kernel when K % 256 == 0, launched with
 * programmatic dependent launch), 1 = always the one-shot split-K kernel, 2 = automatic without
 * programmatic dependent launch, 3 = automatic in EXCLUSIVE mode: the caller vouches that no other kernel holds SMs while a
 * chain runs (one stream, nothing else on the device), and chains with `after` ops are then ordinary launches too (measured:
 * no faster -- cfg2's chain 2.592 vs 2.596 ms, a 25-launch MoE chain 0.4623 vs 0.4623 ms -- so there is no reason to use it); with
 * a foreign kernel on the device such a chain can hang; 4 = automatic without the FUSION of small ops: at batch <= 8 a chain
 * launch deals out independent ops of one shape whose rows are a single chunk (<= 4 KiB: the selected experts' gate, up or down
 * projections of an MoE layer) as one op over all their row tiles, each tile fetched with one bulk copy -- same results bit
 * for bit, 12 Qwen3-MoE-shaped layers 0.477 -> 0.320 ms.  For A/B measurement; process-wide (an atomic: safe to flip from any thread, takes effect at the next
 * launch). */
cloak_status cloak_set_gemv_engine(int engine);
/* Per-SM streaming weights (calibrate.cu): a MEASUREMENT, used by no kernel.  The SMs of a B200 do not pull a read stream out of
 * HBM equally fast (three tiers, up to 1.7 x apart under a dynamic queue, a property of the individual part).  Round 2 cut the
 * streaming GEMV's ops into shares proportional to these weights: 7 % slower (its SMs are limited by their own rings, not by the
 * contended path; equal shares already end together), and the switch alone cost small-op chains 12 %, so it was removed again.
 * cloak_sm_weights: the relative speeds (mean 1) of the device's SMs, indexed by SM id, measured on first use (a 1 GiB scratch
 * buffer, a few ms; synchronises the device); *h_nsm = 0 if they could not be measured.  h_weights may be NULL to query the count. */
cloak_status cloak_sm_weights(int device, uint32_t capacity, float* h_weights, uint32_t* h_nsm);
/* Tracing: while d_trace is not NULL, every streaming-GEMV launch records, per CTA b, four 64-bit words at d_trace[4*b]: the
 * SM id, %globaltimer (ns) at CTA start, when its producer had issued its last copy, and when its consumers were done.  The
 * buffer (DEVICE memory, 8-byte aligned, room for 4 words x the device's SM count) is the caller's and is overwritten by
 * every launch.  NULL switches it off (default).  Process-wide. */
cloak_status cloak_set_trace(void* d_trace);
/* Host only, no device work: the chunk grid one cloak_gemm_chain launch of n_ops <= 16 ops with these shapes would use on a
 * GPU with `sms` SMs under the current cloak_set_gemm_schedule and cloak_set_gemm_engine.  *h_group = g is the number of tile
 * rows a work unit spans (1, or 2 / 4 where the launch groups rows).  The launch's units -- the ops back to back; op j has
 * (N_j / 128 / g) group rows of K_j / 128 units each, unit t of group row R being k step t of tile rows g R .. g R + g - 1 --
 * are numbered 0 .. total-1; chunk c covers units [h_begin[c], h_end[c]).  Chunks 0 .. *h_nstatic-1 are the static shares (CTA c
 * starts with chunk c; a share may be empty), the rest are drawn in order from a counter.  h_begin / h_end may be NULL to query
 * the counts; otherwise they hold max_chunks entries (CLOAK_ERR_INVALID if too few).  Computed by the very functions the
 * kernel calls. */
cloak_status cloak_gemm_plan(uint32_t n_ops, const uint32_t* h_N, const uint32_t* h_K, uint32_t batch, uint32_t sms,
                             uint32_t max_chunks, uint32_t* h_begin, uint32_t* h_end, uint32_t* h_nchunks,
                             uint32_t* h_nstatic, uint32_t* h_group);
/* Schedule of the tcgen05 GEMM: the first `static_pct` percent of a launch's tiles (up to a tile-row boundary) are dealt
 * out in equal shares, one per CTA; the tile rows after that are drawn from a counter as CTAs become free, whole or -- rows
 * of more than `dyn_chunk_tiles` k tiles (0 = by batch) -- in equal pieces.  The chunk grid decides where K is split, so
 * outputs under different settings agree within the bf16 tolerance, not bit for bit; under one setting they do not depend
 * on which CTA drew which chunk.  Default (75, 0).  For A/B measurement; process-wide. */
cloak_status cloak_set_gemm_schedule(int static_pct, int dyn_chunk_tiles);
/* Row groups in the tcgen05 GEMM: 0 = automatic -- at an MMA batch of 32 .. 128 (the caller's batch rounded up to 16), when every
 * matrix of the launch has an even number of 128-row tile rows and the launch holds at least 160 weight tiles per SM (a layer's
 * MLP or more in one chain launch; below that the doubled split-K partials cost more than the X traffic saves, measured),
 * a CTA works on TWO tile rows at a time, which share each X tile (the X
 * traffic out of L2 halves; two accumulator pairs in TMEM: +8-10 % at batch 32 .. 128); 1 = never; 2 = groups of four rows at
 * an MMA batch <= 64 (measured slower than pairs), else pairs, wherever N allows -- whatever the launch size or batch;
 * 3 = pairs wherever N allows.  The grouping changes where K is split, so outputs under different settings agree within the bf16
 * tolerance, not bit for bit.  2 and 3 are for A/B measurement and the tests; process-wide. */
cloak_status cloak_set_gemm_engine(int engine);
/* Host-buffer variant of cloak_gemv (end-to-end path): copies X up, runs, copies Y back, synchronises `stream` once (h_y is
 * the caller's to read on return).  Device staging comes from the library's cached pool: no driver allocation per call. */
cloak_status cloak_gemv_host(const cloak_pool* pool, const cloak_tensor* w, const void* h_x, void* h_y,
                             uint32_t batch, void* stream);

/* Host-buffer form of cloak_gemv_chain for INDEPENDENT ops (no d_gate / d_act / after): every op's d_x and d_y are HOST pointers
 * (pinned for full speed).  All X are copied up, the ops run (one chain launch where the streaming kernel takes them all), all Y
 * are copied back, and `stream` is synchronised once. */
cloak_status cloak_gemv_chain_host(const cloak_pool* pool, const cloak_gemv_op* h_ops, uint32_t n_ops, uint32_t batch,
                                   void* stream);

/* Decode-chain glue: out[i] = silu(g[i]) * u[i] (the gated MLP's activation, O9), n elements. */
cloak_status cloak_silu_mul(const void* d_g, const void* d_u, void* d_out, uint64_t n, cloak_dtype dt,
                            void* stream);

#ifdef __cplusplus
}
#endif
#endif /* CLOAK_H_ */
