/*
 * kinnet.h -- C ABI of the B200 batched explicit-asymptotic network integrator.
 *
 * One opaque net_t holds one reaction network (species/reaction tables, the
 * compiled gather schedule and their device copies).  net_integrate advances
 * `zones` independent copies of that network, each at its own fixed (T9, rho),
 * over one hydro step with the explicit asymptotic method of
 *   Brock, Belt, Billings, Guidry, "Explicit Integration with GPU Acceleration
 *   for Large Kinetic Networks":
 *   Eq. (1)  dy_i/dt = F+_i - F-_i = F+_i - k_i y_i
 *   Eq. (3)  y_n = (y_{n-1} + F+ dt) / (1 + k dt)
 *   branch   k_i dt < kappa -> forward Euler, else Eq. (3)
 *   rates computed once per network integration, fluxes and F+/F- sums every
 *   step, all inside one kernel
 * The adaptive-dt controller and every reading of a point the paper leaves
 * open are in DESIGN.md ("Readings").
 *
 * Conventions
 *   - All functions return NET_OK (0) or a negative NET_E* code; the message is
 *     available from net_last_error() (thread-local).  No exception crosses the
 *     ABI.  Per-zone numerical trouble is reported in status[z], not as a call
 *     failure.
 *   - "host" / "device" below says where a pointer must live.  The caller owns
 *     every array it passes.  net_create copies the host tables; the net_t owns
 *     its device copies and its fixed workspaces.  net_integrate* / net_rates / net_rhs
 *     are asynchronous on `cuda_stream` (a cudaStream_t cast to void*, NULL = default
 *     stream); they allocate nothing, never synchronise, and are legal under stream
 *     capture (every operation they enqueue is a kernel launch or a memset node).
 *   - One net_t may be driven from several streams (and host threads) at once.  The only
 *     per-call device state is the launch-order workspace of net_integrate (4 bytes per
 *     zone + 8 KB): the net_t holds 16 of them ("lanes", 65536 zones each after
 *     net_create, grown by net_reserve) and hands one to every call with >= 1024 zones:
 *       eager calls   the lane the stream used last (stream order serialises its users), else
 *                     a free one, else the least recently used lane whose last zone kernel
 *                     has finished -- streams may come and go, lanes are recycled;
 *       captured calls  a lane of its own per stream capture, never handed out again: the
 *                     graph holds pointers into it and may replay at any time, on any
 *                     stream, beside eager calls and beside other graphs of the same net_t.
 *                     It stays valid until net_destroy.  Every capture that contains a call
 *                     of >= 1024 zones therefore uses up one of the 16 lanes for good.
 *     A call that finds no lane (every lane busy or pinned by a capture, or more zones than
 *     reserved) still runs and returns the same results bit for bit; it only launches the
 *     zones in caller order instead of hottest first (net_launch_stats counts such calls).
 *     No two launches ever share a lane concurrently.  What remains the caller's business:
 *     two replays of the SAME graph must not overlap on the GPU (they would share every
 *     buffer, the lane included), as for any CUDA graph that writes memory.
 *   - A net_t belongs to the CUDA device that was current in net_create; calls with
 *     another device current fail with NET_EINVAL.
 *   - net_integrate_host / net_integrate_host_async take HOST buffers (end to end).
 *   - Y is zone-major [zones * n_species], molar abundances Y_i = X_i / A_i
 *     (Eq. (2) with X the mass fraction); double when the net was
 *     created with precision 64, float with precision 32 (the paper's
 *     single-precision study).
 *   - T9 = T / 1e9 K, rho in g cm^-3, times in s.
 */
#ifndef KINNET_H
#define KINNET_H

#ifdef __cplusplus
extern "C" {
#endif

#define NET_OK 0
#define NET_EINVAL (-1) /* bad argument or table (index out of range, n_react not in 1..3,
                           n_prod not in 1..4, reaction not conserving A, size over limit) */
#define NET_ENOMEM (-2)
#define NET_ECUDA (-3)   /* CUDA runtime error, or no device copy (net_create_host) */

#define NET_MAX_REACT 3
#define NET_MAX_PROD 4
#define NET_N_COEF 7
#define NET_MAX_SPECIES 1024   /* one thread per species, one CTA per zone */
#define NET_MAX_REACTIONS 65535

#define NET_STATUS_MAX_STEPS 1 /* status bit: max_steps sub-steps taken before t_hydro */
#define NET_STATUS_NONFINITE 2 /* status bit: a non-finite abundance was produced    */

typedef struct net net_t;

typedef struct {
    double kappa;        /* branch threshold on k*dt (kappa = 1)            */
    double eps_y;        /* dt control: max relative explicit change per step (0.05)      */
    double y_floor;      /* dt control: abundance floor (1e-10)                           */
    double growth;       /* dt control: dt may grow by at most this factor per step (2)   */
    long long max_steps; /* per call and zone (1e7)                                       */
    int precision;       /* 64 (default) or 32                                            */
    int kernel;          /* 0 = automatic: the two-species-per-thread pull kernel when an instantiation
                            covers the network, else the one-species pull kernel when the network
                            qualifies (every reaction has at most one non-hub reactant, DESIGN.md 4.2;
                            the two-species kernel also takes reactions with two),
                            else the generic flux-array kernel; 1 = always the generic kernel;
                            2 = the one-species pull kernel when the network qualifies (A/B tests) */
    int host_chunk;      /* net_integrate_host*: zones per chunk of the staged path; 0 = default
                            max(16384, zones/16); < 0 = always stage through device scratch, in
                            chunks of -host_chunk zones, even when the buffers are pinned       */
    int method;          /* 0 = the paper's method: Eq. (3) where k dt >= kappa, forward Euler below;
                            1 = explicit quasi-steady-state variant (named as the
                            next step; formula = DESIGN.md reading Q20): every species takes
                            y' = y + dt (F+ - k y) / (1 + alpha(k dt) k dt) with the Pade alpha,
                            behind the same rates, fluxes, sums and dt controller                */
} net_params_t;

/* Fill *p with the defaults listed above. */
int net_default_params(net_params_t *p);

/*
 * Compile a network and upload it to the current CUDA device.
 *   A        host [n_species]      mass numbers
 *   n_react  host [n_reactions]    reactants per reaction, 1..3
 *   react    host [n_reactions*3]  reactant species, repeats allowed, unused = -1
 *   n_prod   host [n_reactions]    products per reaction, 1..4
 *   prod     host [n_reactions*4]  product species, repeats allowed, unused = -1
 *   coef     host [n_reactions*7]  a0..a6 of  ln R = a0 + a1/T9 + a2 T9^(-1/3)
 *                                  + a3 T9^(1/3) + a4 T9 + a5 T9^(5/3) + a6 ln T9
 *   params   host, NULL = defaults
 * The full rate is R = p * rho^(n_react-1) * exp(ln R) with the statistical
 * factor p = 1/prod(m!) over repeated reactants derived here (rate evaluation
 * "from library parameters ... once for each network integration", PAPER.md
 * L104, L197, L202).  This call also builds the host half of the hot path: the
 * flux-slot layout and the deterministic species-to-reaction gather schedule
 * (the flux sums of PAPER.md L197, L215-216; no atomics).
 */
int net_create(net_t **out, int n_species, const int *A, int n_reactions, const int *n_react,
               const int *react, const int *n_prod, const int *prod, const double *coef,
               const net_params_t *params);

/* Same compile without touching CUDA (no device copy; net_integrate* on the
 * result fail with NET_ECUDA).  For schedule inspection on machines without a GPU. */
int net_create_host(net_t **out, int n_species, const int *A, int n_reactions,
                    const int *n_react, const int *react, const int *n_prod, const int *prod,
                    const double *coef, const net_params_t *params);

void net_destroy(net_t *net);

/*
 * One hydro step of length t_hydro for every zone, adaptive network timestep
 * (in = abundances, T, rho, dt_hydro, trial dt;
 * out = abundances, final dt).
 *   T9, rho  device [zones]          held constant over the step (operator split)
 *   Y        device [zones*N]        in/out
 *   dt       device [zones] or NULL  in: trial dt (<= 0 or NULL -> t_hydro);
 *                                    out: last unclamped controller dt
 *   n_steps  device [zones] or NULL  out: sub-steps taken
 *   status   device [zones] or NULL  out: NET_STATUS_* bits
 */
int net_integrate(net_t *net, int zones, const double *T9, const double *rho, void *Y,
                  double t_hydro, double *dt, int *n_steps, int *status, void *cuda_stream);

/*
 * Integrated energy release (the network returns the abundances, the
 * energy released over the hydro step and the final timestep).  The paper gives no formula;
 * DESIGN.md reading Q19: energy[z] = sum_i B_i * (Y_i(t_hydro) - Y_i(0)) with B a per-species
 * binding-energy table supplied by the caller (units: those of B per mole of species, per
 * gram of matter -- e.g. B in MeV gives MeV mol/g; multiply by N_A to get MeV/g).
 *   net_set_binding_energy  B host [n_species]; copied; may be called again to replace it
 *                           (synchronises the device first: a launch in flight may read the table)
 *   net_integrate_energy    net_integrate plus energy device [zones] out (NULL = net_integrate);
 *                           fails with NET_EINVAL if no table has been set
 */
int net_set_binding_energy(net_t *net, const double *B);
int net_integrate_energy(net_t *net, int zones, const double *T9, const double *rho, void *Y,
                         double t_hydro, double *dt, int *n_steps, int *status, double *energy,
                         void *cuda_stream);

/*
 * net_integrate for callers that must not allocate device memory while they run.
 *
 * Who this is for.  net_create reserves the launch-order workspaces of net_integrate with
 * cudaMalloc, and net_reserve grows them the same way.  Some hosts of this library cannot
 * afford that: a hydro code that has handed the whole of HBM to its own pool allocator (a
 * later cudaMalloc fails, or fragments the pool), a code whose time loop lives in a region
 * where the runtime forbids allocation (cudaMalloc synchronises the device and is illegal
 * while a stream is being captured), and real-time or certified drivers in which every byte
 * must be accounted for before the run starts.  For them the one piece of scratch this
 * entry point needs -- the counting sort that launches the hottest zones first (PAPER.md
 * L200 leaves the load balance of unequal networks open) -- lives in a fixed
 * array inside the library image instead of the heap:
 *   (2048 + NET_STATIC_MAX_ZONES) ints = 264 KB of device memory, held by every GPU that
 *   loads libkinnet.so from the moment the CUDA module is loaded until the process exits,
 *   whether or not this function is ever called.
 *
 * Arguments, layouts, units and results are those of net_integrate: the same zone kernel runs
 * on the same inputs, and the order only decides when a zone runs, so the outputs are bit
 * for bit net_integrate's.  The caller still owns and passes every input and output array
 * (device memory).  Differences:
 *   - zones > NET_STATIC_MAX_ZONES fails with NET_EINVAL and a message naming the limit;
 *     nothing is launched.  Split the batch into several calls on ONE stream.
 *   - The call itself performs no cudaMalloc / cudaFree and calls no allocating routine.  It
 *     enqueues a memset of the sort's 8 KB header (counts and cursors must start at zero; the
 *     order itself is fully rewritten by every call, so the previous call's contents never
 *     leak), two small order kernels and the zone kernel on `cuda_stream`, and returns.
 *   - The FIRST call on each device looks the array's device address up
 *     (cudaGetSymbolAddress, with the net_t's device current) and caches it for the life of
 *     the process.  Make that first call at set-up time, before any stream capture begins; a
 *     call with zones = 0 is enough and launches nothing.
 *   - There is ONE array per device, shared by every net_t, stream and host thread.  Two
 *     calls whose GPU work can overlap (calls on different streams with no event between
 *     them, whichever host thread issues them) race on it: zones may then be skipped or
 *     integrated twice.  Issue all calls on a device into one stream, or order them with
 *     events.  net_integrate has per-stream workspaces and no such rule; prefer it
 *     whenever allocation at net_create time is acceptable.
 * The net_t itself is still built by net_create, which allocates its tables: do that during
 * set-up, where allocation is allowed.
 */
#define NET_STATIC_MAX_ZONES 65536
int net_integrate_static(net_t *net, int zones, const double *T9, const double *rho, void *Y,
                         double t_hydro, double *dt, int *n_steps, int *status,
                         void *cuda_stream);

/* Exactly n_steps sub-steps of size dt_fixed for every zone (parity mode).  dt_fixed must be
 * finite and > 0 (NET_EINVAL otherwise). */
int net_integrate_fixed(net_t *net, int zones, const double *T9, const double *rho, void *Y,
                        double dt_fixed, long long n_steps, void *cuda_stream);

/*
 * Grow every launch-order lane to hold max_zones zones (see "Conventions").  Synchronises the
 * device and reallocates: call it at set-up time, never inside a capture or with launches
 * in flight on other host threads.  Shrinks nothing.  Fails with NET_EINVAL (and changes
 * nothing) once a stream capture has taken a lane of this net_t: the captured graph holds
 * pointers into the workspaces this call would free.  Reserve first, capture afterwards.
 */
int net_reserve(net_t *net, int max_zones);

/*
 * Launch-order bookkeeping since net_create (host-side counters; any pointer may be NULL):
 *   sorted_calls    calls of >= 1024 zones that launched hottest first
 *   unsorted_calls  such calls that found no lane and launched in caller order (same bits,
 *                   10-20 % slower on a batch with a wide spread of temperatures)
 *   lanes_pinned    lanes held for good by stream captures, of 16
 */
int net_launch_stats(net_t *net, long long *sorted_calls, long long *unsorted_calls,
                     int *lanes_pinned);

/*
 * End-to-end variants: every array is a HOST buffer -- the 154-in / 152-out float exchange of
 * PAPER.md L106-110, batched (the link and the CPU while the GPU
 * integrates).
 *   - Pinned (page-locked) buffers, e.g. cudaHostAlloc / torch pin_memory: ZERO-COPY.  One
 *     launch over the whole batch; each zone's CTA reads its T9, rho, dt and abundances from the
 *     mapped host buffers when it starts and writes abundances, dt, steps and status back when
 *     it ends, so every transfer overlaps the integration of the other zones and the global
 *     hottest-first order is kept.  No device scratch.
 *   - Any other host memory: staged through device scratch owned by the net_t (grown on
 *     demand: that call then synchronises the internal streams and allocates), in chunks of
 *     params.host_chunk zones over three internal streams; the launch order then applies
 *     within a chunk.  Copies between PAGEABLE memory and the device block the host thread
 *     (an upload until the data are in the driver's staging buffer, a download until it has
 *     finished), so the upload and the kernels of chunk c are enqueued before the download of
 *     chunk c-1: the GPU integrates chunk c while chunk c-1 comes back.  With pageable
 *     buffers net_integrate_host_async therefore returns only when all but the last download
 *     are done; it is asynchronous for pinned buffers (either path).
 *   net_integrate_host_async  enqueues everything and returns; the host buffers must stay
 *                             valid and untouched until net_wait returns.  One batch in
 *                             flight per net_t: a second call before net_wait fails with
 *                             NET_EINVAL and touches nothing.
 *   net_wait                  blocks until the batch enqueued last is back in the host buffers
 *   net_integrate_host        = net_integrate_host_async + net_wait
 * Results are bit for bit those of net_integrate on the same zones, on either path.
 */
int net_integrate_host_async(net_t *net, int zones, const double *T9, const double *rho, void *Y,
                             double t_hydro, double *dt, int *n_steps, int *status);
int net_wait(net_t *net);
int net_integrate_host(net_t *net, int zones, const double *T9, const double *rho, void *Y,
                       double t_hydro, double *dt, int *n_steps, int *status);

/* Rate evaluation alone: R device [zones * n_reactions] (reaction order), double. */
int net_rates(net_t *net, int zones, const double *T9, const double *rho, double *R,
              void *cuda_stream);

/* Fluxes and sums alone for the given state: Fplus, Fminus device [zones*N],
 * same type as Y (Eq. (1) terms). */
int net_rhs(net_t *net, int zones, const double *T9, const double *rho, const void *Y,
            void *Fplus, void *Fminus, void *cuda_stream);

/* Shape of the compiled schedule (all host-side facts). */
typedef struct {
    int n_species, n_reactions;
    int threads;         /* threads per zone (= CTA size), multiple of 32            */
    int flux_slots;      /* flux slots per thread                                    */
    int slots_2body;     /* slots [0, slots_2body) multiply a 2nd reactant           */
    int slots_3body;     /* slots [0, slots_3body) multiply a 3rd reactant           */
    int n_entries;       /* gather entries = sum over reactions of reactants+products */
    int n_big_species;   /* species whose sums are reduced across the CTA            */
    int n_entries_big;   /* entries served by own-slot readback                      */
    int small_max;       /* longest per-thread small-row gather list                 */
    int readback_max;    /* longest per-thread readback list                         */
    int smem_bytes;      /* dynamic shared memory per zone at this precision         */
    int zones_per_sm;    /* co-resident CTAs per SM (0 without a device)             */
    /* the fields above except threads/smem_bytes/zones_per_sm describe the generic
       flux-array schedule; the ones below the pull schedule */
    int kernel;          /* kernel net_integrate* will launch: 0 = generic, 1 = pull (one species
                            per thread), 2 = pull (two species per thread)             */
    int pull_ok;         /* the network qualifies for the pull kernel                 */
    int pull_hubs;       /* hub species tracked in registers by every thread (0..3)   */
    int pull_slots;      /* longest per-thread list of incoming reactions (P-slots)   */
    int pull_slots2;     /* ... of which with a second factor                         */
    int pull_agg_max;    /* longest per-thread rate-sum list                          */
    int pull_wavefronts;       /* predicted shared-memory wavefronts of the fp64 P-slot gathers */
    int pull_wavefronts_ideal; /* ... without bank conflicts                          */
    int pull_threads;    /* (virtual) threads the pull tables are compiled for: = threads for
                            kernel 1, 2 * threads for kernel 2 (a thread plays two of them) */
    int pull_nslots;     /* longest per-thread N-slot list (reactions with two non-hub reactants);
                            0 = the network has none                                    */
    int pull_stair;      /* two-species kernel: 0 = every warp runs the instantiation's slot
                            capacities (always so for blocks of more than 128 threads, i.e. more
                            than 256 species); else bit 0 set = each warp runs its own copy of the sub-step
                            loop, compiled for its step of the staircase of live slots (side a:
                            max(cap_a - 4 w, 12), side b: max(12 - 4 (warps - 1 - w), 4) for warp w);
                            bit 1 = warp 0 plays no species on side b (capacity 0 there); bit 8 + w =
                            warp w's side b does not fit its step and runs the full capacity     */
} net_schedule_info_t;

int net_schedule_info(const net_t *net, net_schedule_info_t *info);

/*
 * Copy one schedule table into out (host, capacity in ints); returns the
 * number of ints the table holds (call with cap = 0 to size), negative on error.
 *   "flux_rxn"    [flux_slots*threads]     reaction of slot j of thread t, -1 = empty
 *   "flux_react"  [flux_slots*threads*3]   its reactant species, n_species = the constant 1
 *   "owner"       [threads]                species owned by thread t, -1 = none
 *   "small_plus"  [threads]                F+ small-row entries of thread t
 *   "small_minus" [threads]                F- small-row entries
 *   "small_src"   [small_max*threads]      entry e of thread t = flux index slot*threads+thread
 *   "big_species" [n_big_species]
 *   "big_cnt"     [2*n_big_species*threads] readback entries of thread t for row 2*s+{0:+,1:-}
 *   "big_slot"    [readback_max*threads]   own flux slot of readback entry e of thread t
 * Pull schedule (only when pull_ok; T = pull_threads, word = index into the published
 * table YP[4][T] followed by the constant one at 4*T):
 *   "pull_hub"      [pull_hubs]            hub species; hub h is owned by thread h
 *   "pull_owner"    [T]                    species owned by thread t, -1 = none
 *   "pull_n_slots"  [T]   "pull_n_slots2" [T]
 *   "pull_slot_rxn" [max(1,pull_slots)*T]  slot e of thread t: reaction | nu << 24, -1 = empty
 *   "pull_slot_f1"  [max(1,pull_slots)*T]  word class*T + thread of its first factor
 *   "pull_slot_f2"  [max(1,pull_slots2)*T] word of its second factor (4*T + 3 = one)
 *   "pull_n_nslots" [T]                    N-slots of thread t: reactions its species enters with
 *                                          another non-hub reactant (k += nu R Y_partner)
 *   "pull_nslot_rxn" [4*T]                 reaction | nu << 24, -1 = empty
 *   "pull_nslot_f1" [4*T]                  word of the partner's abundance
 *   "pull_agg_ptr"  [20*T]                 rate-sum coefficient s of thread t sums entries
 *                                          [ptr[s][t], ptr[s+1][t]) of its list
 *   "pull_agg_ent"  [max(1,pull_agg_max)*T] reaction | nu << 24
 */
int net_schedule_table(const net_t *net, const char *name, int *out, int cap);

const char *net_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* KINNET_H */
