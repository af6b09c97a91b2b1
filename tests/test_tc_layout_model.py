"""Host-side proofs about the tensor kernels (no GPU): what can be shown on the CPU before a launch.

Part A asks the library itself (gmco_tc_schedule: the same tc_layout.h functions the kernels and tc_plan_create
use) for the launch schedule of every shape the host can choose and checks that the shared-memory carve-up fits the
dynamic shared memory that is launched, the TMEM columns fit 512, the ring entries hold their TMA boxes and the TMA
boxes stay inside the global allocations.

Part B is a discrete model of the mbarrier protocols of k_dose_tc, k_dose_tc_pair and k_grad_tc (producer, MMA
issuer, epilogue; ring slot and phase arithmetic, accumulator hand-back parities, arrive counts): under randomly
delayed asynchronous completions (TMA bytes, tcgen05.commit) every configuration must run to completion (no lost
arrival, no wait on a phase that has already gone round twice) and every consumer must find the data it expects in
the slot it reads (no slot overwritten before its MMAs are done, no accumulator reused before it was drained).
The model restates the kernels' index arithmetic by hand; it proves the scheme, the GPU tests prove the code.
"""
import random

import pytest

import paper_1904_01567_b200 as g

K_SLAB, K_TLO, K_PAIR_ENTRY = 16384, 16384, 16384
STRUCTS = (7000, 1600, 1700, 1700)


def _shapes():
    for a in list(range(1, 385, 7)) + [32, 33, 64, 160, 252, 256, 257, 288, 352, 384]:
        for tiles in (1, 2, 3, 4, 7, 8, 9, 16, 31, 32, 33, 79, 80):
            yield a, tiles


@pytest.mark.parametrize("dose_kernel,wide_accum", [(0, 0), (1, 0), (0, 1), (2, 0)])
def test_every_shape_fits_shared_memory_tmem_and_the_allocations(dose_kernel, wide_accum):
    n = 0
    for a, tiles in _shapes():
        for pts in ((64,), (100, 30), STRUCTS, (24000, 4000, 6000, 6000), (40000,)):
            q = g.gmco_tc_schedule(a, pts, 128 * tiles, 148, dose_kernel, wide_accum)
            assert q["ok"] == 1, (a, tiles, pts)
            G = q["a_pad"] // 32
            assert q["a_pad"] == 32 * ((a + 31) // 32) and q["k_pad"] == 128 * tiles and q["n_tiles"] == tiles
            assert q["n_pad"] == sum(64 * ((p + 63) // 64) for p in pts) and q["n_alloc"] % 256 == 0 and q["n_alloc"] >= q["n_pad"]
            # shared memory: carve-up end (from the 1024-aligned base, worst-case alignment loss) <= launched <= opt-in limit
            assert q["dose_smem_end"] + 1023 <= q["dose_smem_bytes"] <= q["smem_limit"] == 227 * 1024
            assert q["grad_smem_end"] + 1023 <= q["grad_smem_bytes"] <= q["smem_limit"]
            assert q["grad_staging_bytes"] == 128 * (q["a_pad"] + 4) * 4 <= q["grad_smem_end"] - 1024
            assert q["grad_stages"] * q["grad_stage_bytes"] <= q["grad_smem_end"] - 1024
            # TMEM
            assert q["dose_tmem_cols"] <= q["tmem_limit"] == 512 and q["grad_tmem_cols"] <= 512
            # ring entries hold their TMA boxes; every operand area starts 1024-aligned (SWIZZLE_128B atoms)
            assert q["dose_stages"] >= 2 and q["grad_stages"] >= 2
            if q["dose_kernel"] in (2, 3):
                assert tiles % 2 == 0 and G <= 8 and dose_kernel in (0, 2)        # any dwell-group count, odd ones included
                assert q["dose_stage_bytes"] == K_PAIR_ENTRY == 32 * 4 * 64 * 2       # box {32 dwell, 64 points, 2 groups}
                assert q["dose_tmem_cols"] == 32 * G + 256
                if q["dose_kernel"] == 2:
                    assert (G + 1) // 2 == 4 and q["dose_stages"] == 6               # 12 entries go twice round a ring of 6
            elif q["dose_kernel"] == 0:
                assert G <= 8 and q["dose_stage_bytes"] == K_SLAB == 32 * 4 * 128     # box {32 dwell, 128 points, 1}
            else:
                assert G > 8 and q["dose_stage_bytes"] == K_SLAB + K_TLO
                assert q["dose_scr_slot"] == q["dose_stages"] - 1                     # the scratch is exactly the last entry
                # T_hi: 8 dwell groups in TMEM + main + corrections, or (wide_accum) 4 groups + two mains + corrections
                assert (q["dose_tmem_groups"], q["dose_n_main"]) == ((4, 2) if wide_accum else (8, 1))
                assert q["dose_tmem_cols"] == 32 * q["dose_tmem_groups"] + 128 * (q["dose_n_main"] + 1) == 512
            if q["dose_kernel"] != 1:
                assert (q["dose_tmem_groups"], q["dose_n_main"]) == (8, 1)            # wide_accum touches the streamed layout only
            assert q["dose_stage_bytes"] % 1024 == 0 and q["grad_stage_bytes"] % 1024 == 0
            if q["grad_pair"]:     # k_grad_tc_pair: each CTA holds its R tile and HALF of the dwell groups of a D slab
                assert dose_kernel == 2 and q["dose_kernel"] in (2, 3) and G % 2 == 0 and q["a_pad"] <= 256 and tiles % 2 == 0
                assert q["grad_stage_bytes"] == 2 * 4 * q["grad_ps"] * 128 + 2 * (G // 2) * q["grad_ps"] * 128
                assert q["grad_tmem_cols"] == 256 + q["a_pad"] <= 512
            else:
                assert dose_kernel != 2 or not (q["dose_kernel"] in (2, 3) and G % 2 == 0)
                assert q["grad_stage_bytes"] == 2 * 4 * q["grad_ps"] * 128 + 2 * G * q["grad_ps"] * 128
            # TMA boxes stay inside the global allocations (rows of D / R: n_alloc; rows of T: k_pad)
            assert q["n_chunks"] * 128 <= q["n_alloc"] and q["n_chunks"] == (q["n_pad"] + 127) // 128
            assert q["n_slabs"] * q["grad_ps"] == q["n_pad"] <= q["n_alloc"]
            assert 1 <= q["segs"] and q["compact_cap"] >= q["segs"]
            n += 1
    assert n > 3000


def test_shapes_outside_the_tensor_route_are_flagged_not_scheduled():
    assert g.gmco_tc_schedule(385, STRUCTS, 1000)["ok"] == 0
    assert g.gmco_tc_schedule(480, STRUCTS, 1000)["ok"] == 0
    with pytest.raises(g.GmcoError):
        g.gmco_tc_schedule(0, STRUCTS, 1000)
    with pytest.raises(g.GmcoError):
        g.gmco_tc_schedule(100, STRUCTS, 0)


def test_split_main_accumulator_flags():
    """gmco_options.wide_accum (k_dose_tc<streamed, split>): a restatement of the issuer's accumulator choice and
    overwrite flags -- per chunk every accumulator is overwritten exactly once, by the first MMA that targets it, the
    overwriting MMA of main accumulator B sits in the shared-memory-tail branch, and the adds split evenly."""
    for G in (9, 10, 11, 12):
        k_tg, g_half = 4, (G + 1) // 2
        log = []                                     # (accumulator, overwrite?, branch) in issue order
        for gq in range(G):
            acc = "A" if gq < g_half else "B"
            first = 0 if gq in (0, g_half) else 1
            branch = "tmem" if gq < k_tg else "tail"
            for j in range(4):
                log.append((acc, (first if j == 0 else 1) == 0, branch))
                log.append(("C", gq == 0 and j == 0, branch))                 # T_lo D_hi
            log += [("C", False, branch)] * 4                                  # T_hi D_lo
        for name in "ABC":
            mine = [x for x in log if x[0] == name]
            assert mine[0][1] and not any(x[1] for x in mine[1:])
        assert [x for x in log if x[0] == "B"][0][2] == "tail"
        nA, nB = sum(x[0] == "A" for x in log), sum(x[0] == "B" for x in log)
        assert nA + nB == 4 * G and abs(nA - nB) <= 4


def test_bench_shapes_take_the_documented_kernels():
    c3 = g.gmco_tc_schedule(252, STRUCTS, 1000)
    assert (c3["dose_kernel"], c3["n_tiles"], c3["segs"], c3["dose_stages"], c3["grad_stages"]) == (2, 8, 18, 6, 4)
    c4 = g.gmco_tc_schedule(384, (24000, 4000, 6000, 6000), 4096)
    assert (c4["dose_kernel"], c4["n_tiles"], c4["segs"]) == (1, 32, 9)
    assert g.gmco_tc_schedule(252, STRUCTS, 1000, dose_kernel=1)["dose_kernel"] == 0
    assert g.gmco_tc_schedule(160, (3500, 800, 850, 850), 100)["dose_kernel"] == 0      # one tile: no pair


# ---------------------------------------------------------------------------------------------------------------------
# Part B: discrete model of the mbarrier protocols
class Bar:
    """mbarrier: `count` arrivals (+ all expected bytes) complete a phase; wait(parity) passes once the phase of that
    parity has completed, i.e. when the parity of the number of completed phases differs from it."""

    def __init__(self, count):
        self.count, self.pending, self.tx, self.phases = count, count, 0, 0

    def _try_complete(self):
        if self.pending == 0 and self.tx == 0:
            self.phases += 1
            self.pending = self.count

    def arrive(self, tx_expect=0):
        assert self.pending > 0, "more arrivals than the barrier's count in one phase"
        self.tx += tx_expect
        self.pending -= 1
        self._try_complete()

    def complete_tx(self, nbytes):
        self.tx -= nbytes
        self._try_complete()

    def passed(self, parity):
        return (self.phases & 1) != parity


class Sim:
    """Round-robin of generator agents with a queue of delayed asynchronous completions."""

    def __init__(self, seed):
        self.rng = random.Random(seed)
        self.pending_async = []       # (due_step, fn)
        self.step = 0

    def later(self, fn):
        self.pending_async.append((self.step + self.rng.randint(0, 12), fn))

    def run(self, agents, limit=2_000_000):
        live = list(agents)
        waits = {}
        while live or self.pending_async:
            self.step += 1
            assert self.step < limit, "model did not terminate"
            due = [x for x in self.pending_async if x[0] <= self.step]
            self.pending_async = [x for x in self.pending_async if x[0] > self.step]
            for _, fn in due:
                fn()
            progressed = bool(due)
            self.rng.shuffle(live)
            for ag in list(live):
                cond = waits.get(id(ag))
                if cond is not None and not cond():
                    continue
                progressed = True
                try:
                    waits[id(ag)] = next(ag)
                except StopIteration:
                    live.remove(ag)
                    waits.pop(id(ag), None)
            if not progressed and not self.pending_async:
                raise AssertionError(f"deadlock: {len(live)} agents wait and nothing is in flight")


def wait(bar, parity):
    return lambda: bar.passed(parity)


def model_dose_single(sim, G, n_stage, n_chunks, resident, scr_slot):
    """k_dose_tc<resident>: ring entries 2g (D_hi [+ T_lo]) and 2g+1 (D_lo) per chunk; one accumulator buffer
    (n_acc = 1); 8 epilogue warps = 256 arrivals hand it back; tg_ready[g]: 128 arrivals of the half of the epilogue
    warps that owns group g."""
    full = [Bar(1) for _ in range(n_stage)]
    empty = [Bar(1) for _ in range(n_stage)]
    tg = [Bar(128) for _ in range(12)]
    tin = [Bar(1) for _ in range(12)]
    acc_full, acc_empty = Bar(1), Bar(256)
    slot_tag = [None] * n_stage
    acc_tag = [None]
    scratch_in_use = [not resident]

    def producer():
        if resident:
            for gq in range(G):
                tin[gq].arrive(K_TLO)
                sim.later(lambda gq=gq: tin[gq].complete_tx(K_TLO))
        st, ph, busy = 0, 0, not resident
        for c in range(n_chunks):
            for g2 in range(2 * G):
                if busy and st >= scr_slot:
                    for i in range(G):
                        yield wait(tg[i], 0)
                    busy = False
                    scratch_in_use[0] = False
                yield wait(empty[st], ph ^ 1)
                if not resident:
                    assert not (scratch_in_use[0] and st >= scr_slot), "TMA into the prologue's scratch"
                nbytes = K_SLAB + (K_TLO if (not resident and g2 % 2 == 0) else 0)
                full[st].arrive(nbytes)

                def land(st=st, c=c, g2=g2, nbytes=nbytes):
                    slot_tag[st] = (c, g2)
                    full[st].complete_tx(nbytes)
                sim.later(land)
                st += 1
                if st == n_stage:
                    st, ph = 0, ph ^ 1

    def issuer():
        st, ph = 0, 0
        for c in range(n_chunks):
            yield wait(acc_empty, (c & 1) ^ 1)
            for gq in range(G):
                for half in range(2):
                    if c == 0 and half == 0:
                        yield wait(tg[gq], 0)
                    yield wait(full[st], ph)
                    assert slot_tag[st] == (c, 2 * gq + half), "issuer read a slot that holds another entry"
                    last = gq == G - 1 and half == 1

                    def done(st=st, c=c, last=last):
                        empty[st].arrive()
                        if last:
                            acc_tag[0] = c
                            acc_full.arrive()
                    sim.later(done)
                    st += 1
                    if st == n_stage:
                        st, ph = 0, ph ^ 1

    def epilogue(h):
        # 4 warps x 32 threads = 128 arrivals per half; prologue: groups h, h + 2, ...
        for gq in range(h, G, 2):
            if resident:
                yield wait(tin[gq], 0)
            for _ in range(128):
                tg[gq].arrive()
            yield None
        for c in range(n_chunks):
            yield wait(acc_full, c & 1)
            assert acc_tag[0] == c, "epilogue read an accumulator of another chunk"
            for _ in range(128):
                acc_empty.arrive()

    sim.run([producer(), issuer(), epilogue(0), epilogue(1)])


def model_dose_pair(sim, G, n_stage, n_chunks, static):
    """k_dose_tc_pair: per chunk 3 Gp entries (2p: D_lo, 2p+1: D_hi corrections; 2Gp+p: D_hi main), two accumulator
    buffers, both CTAs' producers load half of every entry onto the LEADER's full barrier; commits are multicast."""
    Gp = (G + 1) // 2
    E = 3 * Gp
    full = [Bar(1) for _ in range(n_stage)]                      # leader
    empty = [[Bar(1) for _ in range(n_stage)] for _ in range(2)]  # per CTA
    tg = [Bar(256) for _ in range(8)]                            # leader
    tin = [[Bar(1) for _ in range(8)] for _ in range(2)]
    acc_full = [[Bar(1), Bar(1)] for _ in range(2)]
    acc_empty = [Bar(512), Bar(512)]                             # leader
    slot_tag = [[None] * n_stage for _ in range(2)]
    acc_tag = [None, None]

    def producer(rank):
        for gq in range(G):
            tin[rank][gq].arrive(K_TLO)
            sim.later(lambda gq=gq: tin[rank][gq].complete_tx(K_TLO))
        st, ph = 0, 0
        for c in range(n_chunks):
            for g2 in range(E):
                yield wait(empty[rank][st], ph ^ 1)
                if rank == 0:
                    full[st].arrive(2 * K_PAIR_ENTRY)

                def land(st=st, c=c, g2=g2):
                    slot_tag[rank][st] = (c, g2)
                    full[st].complete_tx(K_PAIR_ENTRY)
                sim.later(land)
                st += 1
                if st == n_stage:
                    st, ph = 0, ph ^ 1

    def issuer():
        st, ph, chunk_par = 0, 0, 0
        for c in range(n_chunks):
            b, use = c & 1, c >> 1
            yield wait(acc_empty[b], (use & 1) ^ 1)
            order = []
            for gp in range(Gp):
                order += [(gp, 2 * gp), (gp, 2 * gp + 1)]
            order += [(gp, 2 * Gp + gp) for gp in range(Gp)]
            for gp, e in order:
                if c == 0 and e < 2 * Gp and e % 2 == 0:
                    yield wait(tg[2 * gp], 0)
                    if 2 * gp + 1 < G:
                        yield wait(tg[2 * gp + 1], 0)
                if static:
                    st_e, ph_e = e % n_stage, chunk_par ^ ((e // n_stage) & 1)
                else:
                    st_e, ph_e = st, ph
                yield wait(full[st_e], ph_e)
                for rank in range(2):
                    assert slot_tag[rank][st_e] == (c, e), "issuer read a slot that holds another entry"
                last = e == E - 1

                def done(st_e=st_e, b=b, c=c, last=last):
                    for rank in range(2):
                        empty[rank][st_e].arrive()
                    if last:
                        acc_tag[b] = c
                        for rank in range(2):
                            acc_full[rank][b].arrive()
                sim.later(done)
                st += 1
                if st == n_stage:
                    st, ph = 0, ph ^ 1
            if static:
                assert E % n_stage == 0
                chunk_par ^= (E // n_stage) & 1

    def epilogue(rank, h):
        for gq in range(h, G, 2):
            yield wait(tin[rank][gq], 0)
            for _ in range(128):
                tg[gq].arrive()
            yield None
        for c in range(n_chunks):
            b, use = c & 1, c >> 1
            yield wait(acc_full[rank][b], use & 1)
            assert acc_tag[b] == c, "epilogue read an accumulator of another chunk"
            for _ in range(128):
                acc_empty[b].arrive()

    sim.run([producer(0), producer(1), issuer(), epilogue(0, 0), epilogue(0, 1), epilogue(1, 0), epilogue(1, 1)])


def model_grad(sim, n_stage, n_slabs):
    """k_grad_tc: TMA -> full; 128 converter threads split R in place -> conv; MMA -> empty (commit); last -> acc_full."""
    full = [Bar(1) for _ in range(n_stage)]
    empty = [Bar(1) for _ in range(n_stage)]
    conv = [Bar(128) for _ in range(n_stage)]
    acc_full = Bar(1)
    tag = [None] * n_stage
    split = [None] * n_stage

    def producer():
        st, ph = 0, 0
        for s in range(n_slabs):
            yield wait(empty[st], ph ^ 1)
            full[st].arrive(1000)

            def land(st=st, s=s):
                tag[st] = s
                full[st].complete_tx(1000)
            sim.later(land)
            st += 1
            if st == n_stage:
                st, ph = 0, ph ^ 1

    def converter():
        st, ph = 0, 0
        for s in range(n_slabs):
            yield wait(full[st], ph)
            assert tag[st] == s, "converter read a stage that holds another slab"
            split[st] = s
            for _ in range(128):
                conv[st].arrive()
            st += 1
            if st == n_stage:
                st, ph = 0, ph ^ 1
        if n_slabs:
            yield wait(acc_full, 0)

    def issuer():
        st, ph = 0, 0
        for s in range(n_slabs):
            yield wait(conv[st], ph)
            assert split[st] == s and tag[st] == s, "MMA read a stage that holds another slab"

            def done(st=st, last=(s == n_slabs - 1)):
                empty[st].arrive()
                if last:
                    acc_full.arrive()
            sim.later(done)
            st += 1
            if st == n_stage:
                st, ph = 0, ph ^ 1

    sim.run([producer(), converter(), issuer()])


def test_protocol_model_dose_single_cta_terminates_for_every_host_choice():
    for wide_accum in (0, 1):
        for a_pad in range(32, 385, 32):
            q = g.gmco_tc_schedule(a_pad, STRUCTS, 128, 148, 1, wide_accum)
            assert q["dose_kernel"] in (0, 1)
            G, resident = a_pad // 32, q["dose_kernel"] == 0
            if wide_accum and resident:
                continue
            for n_chunks in (1, 2, 3, 5, 6, 7):
                for seed in range(3):
                    model_dose_single(Sim(seed), G, q["dose_stages"], n_chunks, resident, q["dose_scr_slot"])
    # smaller rings than the host would choose must still be sound (the arithmetic does not depend on a lucky size)
    for G, n_stage in ((8, 2), (8, 3), (5, 4), (1, 2), (3, 7)):
        model_dose_single(Sim(7), G, n_stage, 4, True, -1)
    for G, n_stage in ((9, 2), (12, 3), (10, 5)):
        model_dose_single(Sim(7), G, n_stage, 4, False, n_stage - 1)


def test_protocol_model_dose_cta_pair_terminates_for_every_host_choice():
    for a_pad in (64, 128, 192, 256):
        q = g.gmco_tc_schedule(a_pad, STRUCTS, 256, 148, 0)
        assert q["dose_kernel"] in (2, 3)
        G = a_pad // 32
        for n_chunks in (1, 2, 3, 5, 6, 7):
            for seed in range(3):
                model_dose_pair(Sim(seed), G, q["dose_stages"], n_chunks, q["dose_kernel"] == 2)
    # the kernel also accepts odd group counts (zero-filled half entry) and other ring sizes with the run-time ring
    for G, n_stage in ((7, 6), (7, 5), (3, 2), (1, 2), (5, 12), (8, 5), (8, 12)):
        model_dose_pair(Sim(11), G, n_stage, 5, False)
    model_dose_pair(Sim(11), 7, 6, 5, True)      # static schedule, odd G: GP = 4 entries per pass, last one half-empty


def test_protocol_model_gradient_kernel_terminates_for_every_host_choice():
    for a_pad in range(32, 385, 32):
        q = g.gmco_tc_schedule(a_pad, STRUCTS, 128, 148, 0)
        for n_slabs in (0, 1, 2, q["grad_stages"], q["grad_stages"] + 1, 43):
            for seed in range(3):
                model_grad(Sim(seed), q["grad_stages"], n_slabs)


def test_the_model_does_detect_a_broken_scheme():
    """Sanity of the model itself: a producer that does not wait for `empty` overwrites live slots or loses arrivals."""
    class Lying(Bar):
        def passed(self, parity):
            return True
    with pytest.raises(AssertionError):
        # an accumulator hand-back that nobody waits for: the issuer reuses the buffer before it was drained
        sim = Sim(0)
        full, empty = [Bar(1) for _ in range(2)], [Lying(1) for _ in range(2)]
        tag = [None, None]

        def producer():
            st, ph = 0, 0
            for s in range(8):
                yield wait(empty[st], ph ^ 1)
                full[st].arrive(10)
                sim.later(lambda st=st, s=s: (tag.__setitem__(st, s), full[st].complete_tx(10)))
                st += 1
                if st == 2:
                    st, ph = 0, ph ^ 1

        def consumer():
            st, ph = 0, 0
            for s in range(8):
                yield wait(full[st], ph)
                assert tag[st] == s
                sim.later(lambda st=st: None)
                st += 1
                if st == 2:
                    st, ph = 0, ph ^ 1
        sim.run([producer(), consumer()])
