"""ONE configuration sharded over several GPUs: t-slab decomposition of Algorithm 1.

SURVEY.md section 8(e) / 8(f) NEXT-3; the paper's stated future work (its CPU code does the same
decomposition with PFFT over MPI, :124).  Rank r of N owns the slices t = r T .. (r+1) T - 1 of the lattice.
Every arithmetic step runs in liblgf's kernels through the per-rank entry points ``lgf_slab_*`` (include/lgf.h);
this module only sequences them and moves the buffers between ranks: the F / theta normalisation, the history and
Algorithm 1's loop test are the library's too (``lgf_slab_finalize``, a device-side flag).  The exchanges (the U_t halo only once per
loaded configuration -- the fused sweep keeps it current -- the others once per iteration):

  halo LINKS  U_t of a rank's last slice     -> rank r+1   (a1: A_t(x - t), eq. 5)          S3 * n_l reals
  all-to-all  t-slabs -> z-slabs of F_xyz[Delta]            (a2: the t lines of the 4-D FFT)  8 * V/N * (N-1)/N
              (four of them, one per packed component, each on a second stream while the next component is transformed)
  all-to-all  z-slabs -> t-slabs                            (a4)                              the same
  halo G      g of a rank's first slice      -> rank r-1   (a6: g(x + t), eq. 2)            S3 * 12 reals
  halo G_UP   g of a rank's last slice       -> rank r+1   (fused a6 + a1: g(x - t))        S3 * 12 reals
  all-reduce  (sum Re tr U, sum tr Delta Delta^dag)         (F, theta, eqs. 3, 6)             2 doubles

Two exchange objects implement them:

* ``DistExchange``: one process per GPU, torch.distributed (NCCL over NVLink / NVSwitch: batched isend / irecv for
  the halos, ``all_to_all_single`` for the transposition, ``all_reduce`` for the sums).  On gloo it moves CPU
  tensors the same way (tests/test_slab_gloo.py, world_size 2).
* ``LocalExchange``: all N ranks emulated in ONE process on one GPU.  Each phase is run for every rank in turn and
  the exchange is a set of device copies between the ranks' buffers, so no kernel ever waits on another rank
  (B200_PROFILING.md: emulate ranks as successive launches over all ranks' data, never as concurrently waiting
  kernels).  This is how the path is checked against the oracle on the one-GPU box (tests/test_gpu_slab.py).

Both have the same three methods over LISTS of per-local-rank tensors (length N for LocalExchange, 1 for
DistExchange), so ``SlabFixer`` is the same code in both cases.  No CPU fallback: the kernels need liblgf.so and
a CUDA device.  This module never touches the oracle.
"""
from __future__ import annotations

from typing import List, Sequence

from . import binding as B


NCOMP = 4       # packed components of the work field: the all-to-all buffers are [c][q][tl][zl][y][x] (include/lgf.h)


class LocalExchange:
    """N ranks emulated in one process (see module docstring)."""

    def __init__(self, world: int):
        if world < 1:
            raise ValueError("world must be >= 1")
        self.world = int(world)
        self.local_ranks = list(range(self.world))

    def shift(self, send: Sequence, recv: Sequence, step: int) -> None:
        """recv[r] <- send[(r - step) mod N]: every rank sends to rank r + step."""
        n = self.world
        for r in range(n):
            recv[r].copy_(send[(r - step) % n])

    def all_to_all_comp(self, send: Sequence, recv: Sequence, c: int) -> None:
        """Component c's quarter of the buffers: chunk q of rank r's quarter becomes chunk r of rank q's (equal chunks)."""
        n = self.world
        for r in range(n):
            dst = recv[r].view(NCOMP, n, -1)[c]
            for q in range(n):
                dst[q].copy_(send[q].view(NCOMP, n, -1)[c][r])

    def all_to_all(self, send: Sequence, recv: Sequence) -> None:
        for c in range(NCOMP):
            self.all_to_all_comp(send, recv, c)

    # the overlapped form: here the "exchange" is device copies in stream order, so start = do it, finish = nothing
    def start_all_to_all_comp(self, send, recv, c, main=None, comm=None):
        self.all_to_all_comp(send, recv, c)
        return None

    def finish(self, handle, main=None) -> None:
        return None

    def all_reduce_sum(self, vals: Sequence) -> None:
        total = vals[0].clone()
        for v in vals[1:]:
            total += v                      # fixed order: rank 0, 1, ..., N-1
        for v in vals:
            v.copy_(total)


class DistExchange:
    """One process per rank over torch.distributed (nccl on the GPUs, gloo on the CPU)."""

    def __init__(self, dist, group=None):
        self.dist, self.group = dist, group
        self.world = dist.get_world_size(group)
        self.rank = dist.get_rank(group)
        self.local_ranks = [self.rank]

    def _global(self, r: int) -> int:
        return r if self.group is None else self.dist.get_global_rank(self.group, r)

    def shift(self, send, recv, step: int) -> None:
        n, r, dist = self.world, self.rank, self.dist
        if n == 1:
            recv[0].copy_(send[0])
            return
        ops = [dist.P2POp(dist.isend, send[0], self._global((r + step) % n), self.group),
               dist.P2POp(dist.irecv, recv[0], self._global((r - step) % n), self.group)]
        for w in dist.batch_isend_irecv(ops):
            w.wait()

    def all_to_all_comp(self, send, recv, c: int, async_op: bool = False):
        s, r = send[0].view(NCOMP, -1)[c], recv[0].view(NCOMP, -1)[c]
        if self.world == 1:
            r.copy_(s)
            return None
        return self.dist.all_to_all_single(r, s, group=self.group, async_op=async_op)

    def all_to_all(self, send, recv) -> None:
        for c in range(NCOMP):
            self.all_to_all_comp(send, recv, c)

    def start_all_to_all_comp(self, send, recv, c: int, main=None, comm=None):
        """Component c's exchange on the stream `comm`, after what `main` has enqueued so far; returns a handle for
        ``finish``.  While it runs, `main` is free for the next component's kernels.  CPU tensors (gloo): done here."""
        if not send[0].is_cuda or comm is None:
            self.all_to_all_comp(send, recv, c)
            return None
        import torch

        ev = torch.cuda.Event()
        ev.record(main)
        comm.wait_event(ev)
        with torch.cuda.stream(comm):
            work = self.all_to_all_comp(send, recv, c, async_op=True)      # None for one rank: a copy on `comm`
            done = torch.cuda.Event()
            done.record(comm)
        return (work, done)

    def finish(self, handle, main=None) -> None:
        """Makes `main` wait (on the device, not the host) for the exchange started with ``start_all_to_all_comp``."""
        if handle is None:
            return
        import torch

        work, done = handle
        with torch.cuda.stream(main):
            if work is not None:
                work.wait()                  # NCCL: the current stream waits for the collective
            main.wait_event(done)

    def all_reduce_sum(self, vals) -> None:
        if self.world > 1:
            self.dist.all_reduce(vals[0], group=self.group)


def slab_of(links, rank: int, world: int):
    """Rank `rank`'s t-slab of a canonical configuration [Lt, Lz, Ly, Lx, 4, 3, 3(, 2)] (a contiguous slice)."""
    Lt = links.shape[0]
    if Lt % world:
        raise ValueError("world must divide Lt")
    T = Lt // world
    return links[rank * T:(rank + 1) * T]


class SlabFixer:
    """Algorithm 1 on one configuration sharded over ``exchange.world`` ranks.

    dims = GLOBAL (Lx, Ly, Lz, Lt); world must divide Lt and Lz.  History entry n = (F, theta) of the configuration
    after n updates since ``set_links`` (as lgf_iterate / lgf_fix, include/lgf.h)."""

    def __init__(self, dims, precision=B.LGF_FP64, link_storage=B.LGF_LINKS_18, exchange=None, device=None, overlap=None):
        import torch

        self.torch = torch
        self.ex = exchange if exchange is not None else LocalExchange(1)
        self.dims = tuple(int(v) for v in dims)
        self.precision, self.link_storage = int(precision), int(link_storage)
        self.device = torch.device(device) if device is not None else torch.device("cuda", torch.cuda.current_device())
        self.V = self.dims[0] * self.dims[1] * self.dims[2] * self.dims[3]
        world = self.ex.world
        stream = torch.cuda.current_stream(self.device)
        self.ranks: List[B.SlabContext] = [B.SlabContext(self.dims, precision, link_storage, r, world, stream=stream)
                                           for r in self.ex.local_ranks]
        rdt = torch.float64 if precision == B.LGF_FP64 else torch.float32
        mk = lambda n, dt=rdt: [torch.empty(n, dtype=dt, device=self.device) for _ in self.ranks]
        c0 = self.ranks[0]
        self._u_send, self._u_recv = mk(c0.halo_elems(B.LGF_HALO_LINKS)), mk(c0.halo_elems(B.LGF_HALO_LINKS))
        self._g_send, self._g_recv = mk(c0.halo_elems(B.LGF_HALO_G)), mk(c0.halo_elems(B.LGF_HALO_G))
        self._g2_send, self._g2_recv = mk(c0.halo_elems(B.LGF_HALO_G_UP)), mk(c0.halo_elems(B.LGF_HALO_G_UP))
        self._a_send, self._a_recv = mk(c0.V * 8), mk(c0.V * 8)
        self._sums = mk(2, torch.float64)
        # overlap of the exchanges with the line passes: component c's all-to-all on a second stream while component
        # c + 1 is transformed (needs the per-component entry points; `overlap=False` keeps the plain order)
        # overlap=None: only with more than one rank -- with one rank there is nothing to hide and the 12 smaller
        # launches cost 8 % (32^4 fp64 on one B200: 0.535 against 0.497 ms per iteration)
        if overlap is None:
            overlap = world > 1
        self.overlap = bool(overlap) and all(c.by_component() for c in self.ranks)
        self._main = stream
        self._comm = torch.cuda.Stream(self.device) if self.overlap else None
        self._w_is_delta = False        # W of every rank holds Delta of the current links (and _sums their all-reduced sums)
        self._recorded = False          # ... and that configuration's (F, theta) is in the history
        self.exchanged_bytes = 0        # per rank, what the last iterate() sent (bench / DESIGN.md figures)

    # -- configuration ----------------------------------------------------------------------------
    def set_links(self, slabs: Sequence) -> None:
        """One canonical slab per local rank ([T, Lz, Ly, Lx, 4, 3, 3, 2] real or [..., 3, 3] complex, on the device)."""
        if len(slabs) != len(self.ranks):
            raise ValueError("expected %d slab(s)" % len(self.ranks))
        for c, s in zip(self.ranks, slabs):
            c.set_links(s.contiguous())
        self._w_is_delta, self._recorded = False, False

    def set_links_global(self, links) -> None:
        self.set_links([slab_of(links, r, self.ex.world) for r in self.ex.local_ranks])

    def get_links(self) -> list:
        rdt = self.torch.float64 if self.precision == B.LGF_FP64 else self.torch.float32
        out = []
        for c in self.ranks:
            t = self.torch.empty((c.T, self.dims[2], self.dims[1], self.dims[0], 4, 3, 3, 2), dtype=rdt, device=self.device)
            out.append(c.get_links(t))
        return out

    # -- the steps of one iteration ---------------------------------------------------------------
    def _step_delta(self, tol: float, record: bool) -> None:
        """a1 (+ halo of U_t, all-reduce of the sums, finalize on the device): Delta into every rank's work field;
        F, theta into the state, and with `record` into the history together with the loop test theta < tol."""
        for c, s in zip(self.ranks, self._u_send):
            c.halo_pack(B.LGF_HALO_LINKS, s)
        self.ex.shift(self._u_send, self._u_recv, +1)
        for c, r, sm in zip(self.ranks, self._u_recv, self._sums):
            c.halo_unpack(B.LGF_HALO_LINKS, r)
            c.delta(sm)
        self.ex.all_reduce_sum(self._sums)
        for c, sm in zip(self.ranks, self._sums):
            c.finalize(sm, tol, False, record)
        self._w_is_delta = True
        self._recorded = self._recorded or record

    def _fft_by_component(self) -> None:
        """a2-a4 up to the work field in (x, y) k space, one packed component at a time: while component c's all-to-all
        runs on the second stream, the main stream already transforms component c + 1.  Per component the order is
        forward x, y, z -> exchange 1 -> t lines (forward, scale, inverse) -> exchange 2 -> inverse z; buffers: the
        t pass of c reads recv[c] and refills send[c] (its first exchange is over), the second exchange refills recv[c]
        (its t pass is over) -- each ordered by the handle of the step before."""
        ex, main, comm = self.ex, self._main, self._comm
        first, second = [], []
        for k in range(NCOMP):
            for c, s in zip(self.ranks, self._a_send):
                c.fft_forward_comp(s, k)
            first.append(ex.start_all_to_all_comp(self._a_send, self._a_recv, k, main, comm))
        for k in range(NCOMP):
            ex.finish(first[k], main)
            for c, s, r in zip(self.ranks, self._a_send, self._a_recv):
                c.fft_t_comp(r, s, k)
            second.append(ex.start_all_to_all_comp(self._a_send, self._a_recv, k, main, comm))
        for k in range(NCOMP):
            ex.finish(second[k], main)
            for c, r in zip(self.ranks, self._a_recv):
                c.fft_zinv_comp(r, k)

    def _fft_to_second_exchange(self) -> None:
        for c, s in zip(self.ranks, self._a_send):
            c.fft_forward(s)
        self.ex.all_to_all(self._a_send, self._a_recv)
        for c, s, r in zip(self.ranks, self._a_send, self._a_recv):
            c.fft_t(r, s)
        self.ex.all_to_all(self._a_send, self._a_recv)

    def _step_accelerate(self) -> None:
        """a2-a4: w = F^-1[(p2max / p2) F Delta] / V with the t lines gathered by two all-to-alls; w into the work field."""
        if self.overlap:
            self._fft_by_component()
            for c in self.ranks:
                c.fft_xyinv(False)
            return
        self._fft_to_second_exchange()
        for c, r in zip(self.ranks, self._a_recv):
            c.fft_inverse(r)

    def _step_update(self, alpha: float, g_ready: bool = False) -> None:
        """a5 + a6 (+ halo of g)."""
        for c, s in zip(self.ranks, self._g_send):
            if not g_ready:
                c.gbuild(alpha)
            c.halo_pack(B.LGF_HALO_G, s)
        self.ex.shift(self._g_send, self._g_recv, -1)
        for c, r in zip(self.ranks, self._g_recv):
            c.halo_unpack(B.LGF_HALO_G, r)
            c.update()
        self._w_is_delta, self._recorded = False, False

    def _step_iteration(self, alpha: float, tol: float) -> None:
        """a2-a6 + a1 of the new links, as iterate / fix run them: the g-build at the end of the last FFT sweep, g halos
        both ways, the fused sweep (new links, their Delta and sums in one pass), all-reduce, finalize on the device
        (new buffer current, history, loop test).  Wants the work fields to hold Delta of the current links, which
        also means the U_t halos are current.  Nothing is read back: once the device-side `done` flag is set the
        kernels of later iterations return at once."""
        if self.overlap:
            self._fft_by_component()
        else:
            self._fft_to_second_exchange()
        for c, r, dn, up in zip(self.ranks, self._a_recv, self._g_send, self._g2_send):
            if self.overlap:
                c.fft_xyinv(True, alpha)
            else:
                c.fft_inverse_g(r, alpha)
            c.halo_pack(B.LGF_HALO_G, dn)
            c.halo_pack(B.LGF_HALO_G_UP, up)
        self.ex.shift(self._g_send, self._g_recv, -1)
        self.ex.shift(self._g2_send, self._g2_recv, +1)
        for c, dn, up, sm in zip(self.ranks, self._g_recv, self._g2_recv, self._sums):
            c.halo_unpack(B.LGF_HALO_G, dn)
            c.halo_unpack(B.LGF_HALO_G_UP, up)
            c.sweep(sm)
        self.ex.all_reduce_sum(self._sums)
        for c, sm in zip(self.ranks, self._sums):
            c.finalize(sm, tol, True, True)
        self._w_is_delta, self._recorded = True, True

    def _bytes_per_iteration(self) -> int:
        n, es = self.ex.world, self._a_send[0].element_size()
        if n == 1:
            return 0
        a2a = 2 * self._a_send[0].numel() * es * (n - 1) // n
        return a2a + (self._g_send[0].numel() + self._g2_send[0].numel()) * es + 16

    # -- public: same meaning as lgf_measure / lgf_iterate / lgf_fix ---------------------------------
    def _look(self):
        """(done, nan, n_updates, F, theta) as the device state stands after everything enqueued so far."""
        for c in self.ranks:
            c.poll()
        return [c.poll_wait() for c in self.ranks][0]

    def _first_measure(self, tol: float) -> None:
        """Alg. 1 line 1: Delta, F, theta of the loaded configuration as history entry 0, with the first loop test."""
        if not (self._w_is_delta and self._recorded):
            self._step_delta(tol, True)

    def measure(self):
        """(F, theta) of the current configuration (eqs. 3, 6), computed by the library; records nothing; synchronises."""
        self._step_delta(-1.0, False)
        _, _, _, F, theta = self._look()
        return F, theta

    def iterate(self, alpha: float, n: int) -> None:
        """n updates regardless of theta; leaves n + 1 history entries from a fresh configuration.  Never reads
        a value back to the host."""
        for c in self.ranks:
            c.clear_done()
        self._first_measure(-1.0)
        for _ in range(int(n)):
            self._step_iteration(alpha, -1.0)
        self.exchanged_bytes = self._bytes_per_iteration() * int(n)

    def fix(self, alpha: float, tol: float, max_iter: int, chunk: int = 16) -> int:
        """measure; while theta >= tol and it < max_iter: update; measure (Alg. 1).  Returns the number of updates.
        The loop test is taken on the device (lgf_slab_finalize); the host enqueues `chunk` iterations at a time and
        looks at the state one chunk behind, so the GPU never waits for the host."""
        for c in self.ranks:
            c.clear_done()
        self._first_measure(tol)
        issued, outstanding, done = 0, 0, False
        while not done and issued < max_iter:
            n = min(chunk, max_iter - issued)
            for _ in range(n):
                self._step_iteration(alpha, tol)
            issued += n
            for c in self.ranks:
                c.poll()
            outstanding += 1
            if outstanding >= 2:            # the look taken one chunk ago; the chunk just enqueued keeps the GPU busy
                done = [c.poll_wait() for c in self.ranks][0][0]
                outstanding -= 1
        while outstanding:
            for c in self.ranks:
                c.poll_wait()
            outstanding -= 1
        done, nan, updates, _, _ = self._look()
        if nan:
            raise B.LgfError(B.LGF_ENAN, "theta became NaN")
        return updates

    def history(self):
        """(F[], theta[]) numpy arrays of the recorded entries (every rank holds the same); synchronises."""
        return self.ranks[0].history()

    @property
    def updates(self) -> int:
        return self._look()[2]

    def work_field(self) -> list:
        """Every local rank's work field (Delta after a measurement) as [T, Lz, Ly, Lx, 3, 3, 2] tensors."""
        rdt = self.torch.float64 if self.precision == B.LGF_FP64 else self.torch.float32
        out = []
        for c in self.ranks:
            t = self.torch.empty((c.T, self.dims[2], self.dims[1], self.dims[0], 3, 3, 2), dtype=rdt, device=self.device)
            out.append(c.get_field(t))
        return out

    def launch_count(self) -> int:
        return sum(c.launch_count() for c in self.ranks)

    def destroy(self) -> None:
        for c in self.ranks:
            c.destroy()
        self.ranks = []
