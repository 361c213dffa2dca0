"""Stage-per-GPU PACI: rank s of a `torch.distributed` job holds stage s on its own B200 and runs
Algorithm 1's LOCAL event loop; the only traffic is point to point between neighbours --
h_{m,i} forward (Alg. 1 line 8) and grad h_{m,i-1} backward (line 14), [mu, T, D] in the
compute dtype.  No collective, no barrier between stages, no global step.

What is different from the one-GPU schedule driver (`paci_pipeline_run`): there the S stages are streams of one
device in a canonical LOGICAL schedule, so crossed-update counts are reproducible and compared exactly with the
oracle; here every stage really is asynchronous ("stages execute ... independently as soon as the required input
tensors arrive"), the order of events depends on arrival times, and what holds is the paper's BOUND
Delta_{m,i} <= ceil((N - i) / a) (Eq. 2 / Eq. 10, "without relying on balanced stage times") -- the
tests check the bound, the admission cap and the FIFO order, not one particular interleaving.

Transport.  One 2-rank process group per boundary AND direction (NCCL: its own communicator and stream), so a stage's
pending receive of the next activation never sits in front of its send of a gradient on the same stream (with a single
communicator the two neighbours' sends would wait for each other's receives).  Receives are posted ahead into a ring of
`depth` buffers per direction; a message is consumed in micro-batch order (all queues are FIFO, R4).  Over
NVLink 5 / NVSwitch the 16.8 MB boundary tensor of configs[2] takes ~22 us at the measured 770 GB/s, against stage steps
of several milliseconds, and NCCL issues it on its own stream, so it overlaps the next kernels of the stage.

The stage object is anything with the `binding.Stage` interface (forward, backward, maybe_step, unresolved,
crossed_updates, version): the CPU tests drive this module over gloo with a stand-in; on GPUs it is `binding.Stage`.
This module is host-side plumbing only: every step of the path runs in the library's kernels.
"""
from __future__ import annotations

import time


class BoundaryGroups:
    """groups[(s, 'f')] carries h from rank s to s + 1, groups[(s, 'b')] carries grad h from s + 1 to s.
    Every rank must construct this (new_group is collective) in the same order."""

    def __init__(self, world_size: int):
        import torch.distributed as dist
        self.groups = {}
        for s in range(world_size - 1):
            for d in ("f", "b"):
                self.groups[(s, d)] = dist.new_group([s, s + 1])


class _Inbox:
    """Messages 0 .. n-1 from one neighbour, in order, into a ring of `depth` buffers.  ready(m) never blocks.

    NCCL: receives are posted ahead with irecv and `is_completed()` is a CUDA-event query.  gloo (the CPU tests): a
    Work's `is_completed()` stays false until someone waits on it, and a wait with a timeout tears the pair down, so a
    daemon thread does blocking receives into the free ring slots and publishes how many have landed."""

    def __init__(self, bufs, src, group, n):
        import threading
        import torch.distributed as dist
        self.bufs, self.src, self.group, self.n, self.R = bufs, src, group, n, len(bufs)
        self.consumed = 0
        self.threaded = dist.get_backend(group) != "nccl"
        if self.threaded:
            self.arrived = 0
            self.cv = threading.Condition()
            self.error = None
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        else:
            self.reqs, self.posted = {}, 0
            self._post()

    def _pump(self):
        import torch.distributed as dist
        try:
            for m in range(self.n):
                with self.cv:
                    self.cv.wait_for(lambda: m < self.consumed + self.R)      # ring slot free
                dist.recv(self.bufs[m % self.R], src=self.src, group=self.group)
                with self.cv:
                    self.arrived = m + 1
        except Exception as e:                                               # surfaced by ready()
            self.error = e

    def _post(self):
        import torch.distributed as dist
        while self.posted < self.n and self.posted < self.consumed + self.R:
            self.reqs[self.posted] = dist.irecv(self.bufs[self.posted % self.R], src=self.src, group=self.group)
            self.posted += 1

    def ready(self, m):
        if self.threaded:
            if self.error is not None:
                raise self.error
            return self.arrived > m
        return self.reqs[m].is_completed()

    def take(self, m):
        """The buffer holding message m (which must be ready)."""
        if not self.threaded:
            self.reqs.pop(m).wait()
        return self.bufs[m % self.R]

    def release(self, m):
        """Message m has been consumed (the work reading it is enqueued): its ring slot may be refilled."""
        if self.threaded:
            with self.cv:
                self.consumed = m + 1
                self.cv.notify_all()
        else:
            self.consumed = m + 1
            self._post()


class _Outbox:
    """Sends in order out of a ring of `depth` buffers; a slot is rewritten only after its last send completed."""

    def __init__(self, bufs, dst, group):
        self.bufs, self.dst, self.group, self.R, self.reqs = bufs, dst, group, len(bufs), {}

    def buffer(self, m):
        req = self.reqs.pop(m - self.R, None)
        if req is not None:
            req.wait()
        return self.bufs[m % self.R]

    def send(self, m):
        import torch.distributed as dist
        self.reqs[m] = dist.isend(self.bufs[m % self.R], dst=self.dst, group=self.group)

    def drain(self):
        for req in self.reqs.values():
            req.wait()
        self.reqs.clear()


class StageWorker:
    """Algorithm 1 for ONE stage.  `make_buffer()` returns an empty boundary tensor [mu, T, D] on the stage's device."""

    def __init__(self, stage, stage_index: int, n_stages: int, make_buffer, groups: BoundaryGroups | None,
                 depth: int | None = None):
        self.stage, self.s, self.S = stage, stage_index, n_stages
        self.groups = groups.groups if groups is not None else {}
        self.depth = depth if depth is not None else n_stages      # messages that may be in flight per direction
        first, last = stage_index == 0, stage_index == n_stages - 1
        self.fwd_in = None if first else [make_buffer() for _ in range(self.depth)]
        self.bwd_in = None if last else [make_buffer() for _ in range(self.depth)]
        self.fwd_out = None if last else [make_buffer() for _ in range(self.depth)]
        self.bwd_out = None if first else [make_buffer() for _ in range(self.depth)]

    def run(self, n_microbatches: int, lr, inputs=None, targets=None, losses=None, poll_sleep: float = 0.0):
        """Processes micro-batches 0 .. n-1.  inputs(m) -> int32 tokens [mu, T] (stage 0 only); targets(m) -> int32
        [mu, T] and losses[m] a float[1] device buffer (last stage only); lr: float or callable(local update index).
        Returns dict(delta=[...], version, max_q, events=[('F'|'B'|'U', m), ...])."""
        st, s, S, n = self.stage, self.s, self.S, n_microbatches
        first, last = s == 0, s == S - 1
        cap = S - 1 - s                                           # Eq. 9: admit a forward iff q <= N - i
        g = self.groups
        f_in = None if first else _Inbox(self.fwd_in, s - 1, g[(s - 1, "f")], n)
        b_in = None if last else _Inbox(self.bwd_in, s + 1, g[(s, "b")], n)
        f_out = None if last else _Outbox(self.fwd_out, s + 1, g[(s, "f")])
        b_out = None if first else _Outbox(self.bwd_out, s - 1, g[(s - 1, "b")])
        nf = nb = 0                                               # next forward / next backward (FIFO)
        delta, events, max_q = [], [], 0
        lr_of = lr if callable(lr) else (lambda t: lr)
        while nb < n:
            b_ready = nb < nf and (last or b_in.ready(nb))
            f_ready = nf < n and st.unresolved <= cap and (first or f_in.ready(nf))
            if b_ready:                                           # a ready backward goes first (R1)
                m = nb
                dout = None if last else b_in.take(m)
                din = None if first else b_out.buffer(m)
                st.backward(m, dout, din)                         # stashed activations, CURRENT weights (Eq. 1)
                if not last:
                    b_in.release(m)
                if not first:
                    b_out.send(m)
                delta.append(st.crossed_updates(m))               # Eq. 8, read before the update test
                events.append(("B", m))
                if st.maybe_step(lr_of(st.version)):              # Alg. 1 lines 16-19
                    events.append(("U", st.version))
                nb += 1
            elif f_ready:
                m = nf
                inp = inputs(m) if first else f_in.take(m)
                out = losses[m] if last else f_out.buffer(m)
                st.forward(m, inp, targets(m) if last else None, out)
                if not first:
                    f_in.release(m)
                if not last:
                    f_out.send(m)
                events.append(("F", m))
                nf += 1
                max_q = max(max_q, st.unresolved)
            elif poll_sleep > 0.0:
                time.sleep(poll_sleep)
        for box in (f_out, b_out):
            if box is not None:
                box.drain()
        return dict(delta=delta, version=st.version, max_q=max_q, events=events)
