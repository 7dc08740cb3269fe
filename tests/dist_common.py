"""Several ranks of paper_2606_12650_b200.dist inside ONE process (one GPU): every rank is a host thread
running the same SPMD code as under torchrun; the communicator's all-gather and neighbour exchange are device copies
between the ranks' buffers, ordered by stream synchronisation and a host barrier (no kernel waits on another)."""
import threading


class _Shared:
    def __init__(self, world):
        self.world = world
        self.barrier = threading.Barrier(world, timeout=300)
        self.slots = [None] * world


class ThreadComm:
    def __init__(self, shared, rank):
        self._sh, self.rank, self.world = shared, rank, shared.world

    def all_gather_object(self, obj):
        sh = self._sh
        sh.slots[self.rank] = obj
        sh.barrier.wait()
        out = list(sh.slots)
        sh.barrier.wait()
        return out

    def all_gather(self, send, out):
        import torch
        sh = self._sh
        if send.is_cuda:
            torch.cuda.synchronize()
        sh.slots[self.rank] = send
        sh.barrier.wait()
        rows = out.view(self.world, -1)
        for r in range(self.world):
            rows[r].copy_(sh.slots[r])
        if send.is_cuda:
            torch.cuda.synchronize()
        sh.barrier.wait()


    def exchange(self, send, recv, neighbours):
        """Segment [off, off + cnt) of `send` to, and of `recv` from, every neighbour: device copies between the ranks'
        buffers (each rank publishes its buffer and where each neighbour's segment sits in it)."""
        import torch
        sh = self._sh
        if send.is_cuda:
            torch.cuda.synchronize()
        sh.slots[self.rank] = (send, {r: (off, cnt) for r, off, cnt in neighbours})
        sh.barrier.wait()
        for r, off, cnt in neighbours:
            theirs, table = sh.slots[r]
            toff, tcnt = table[self.rank]
            assert tcnt == cnt, "the two ranks disagree on how many nodes they share"
            recv[off:off + cnt].copy_(theirs[toff:toff + tcnt])
        if send.is_cuda:
            torch.cuda.synchronize()
        sh.barrier.wait()


def run_ranks(world, fn):
    """fn(comm) on `world` threads; returns the list of results by rank, re-raises the first failure."""
    sh = _Shared(world)
    res, err = [None] * world, [None] * world

    def body(r):
        try:
            res[r] = fn(ThreadComm(sh, r))
        except BaseException as e:          # noqa: BLE001 - reported below
            err[r] = e
            sh.barrier.abort()

    ts = [threading.Thread(target=body, args=(r,)) for r in range(world)]
    for t in ts:
        t.start()
    for t in ts:
        t.join()
    real = [e for e in err if e is not None and not isinstance(e, threading.BrokenBarrierError)]
    if real or any(err):
        raise (real[0] if real else next(e for e in err if e is not None))
    return res
