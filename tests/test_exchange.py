"""paper_1704_00513_b200/exchange.py (Algorithm 4): the frontier exchange of a
BFS level with the codec on both sides.
CPU (not gpu): the host logic of PackedExchange on a 2-rank gloo group, with a codec object made from the ORACLE (test-only
injection: the product's codec is the CUDA binding and has no CPU path), and the slot address arithmetic.
GPU: SlotExchange with four ranks' buffers on one device (each rank's call sequence run in turn: no kernel waits for
another), SlotExchange over real symmetric memory and PackedExchange over NCCL in a 1-rank group. Expected result in all
cases: rank d receives from rank s exactly the list s held for d (integer work: bit-exact), and every stream on the wire
is the oracle's stream of that list."""
import os

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def level_buffers(level, src, P, W, n_vertices=1 << 22, dense=False):
    """What rank `src` found for every owner d at `level`: ascending unique IDs inside d's vertex range (seeded by
    level / src / d; some buffers empty, sizes from a handful to tens of thousands)."""
    chunk = n_vertices // P
    lists = []
    for d in range(P):
        g = torch.Generator().manual_seed(1000 * level + 37 * src + d)
        n = int(torch.randint(0, 40000 if dense else 3000, (1,), generator=g))
        if (level + src + d) % 5 == 0:
            n = 0
        if (level + src + d) % 7 == 1:
            n = 3
        v = torch.randperm(chunk, generator=g)[:n].sort().values + d * chunk
        lists.append(v)
    counts = torch.tensor([len(v) for v in lists], dtype=torch.int64)
    off = torch.zeros(P + 1, dtype=torch.int64)
    off[1:] = torch.cumsum(counts, 0)
    ids = torch.cat(lists) if P else torch.zeros(0, dtype=torch.int64)
    return ids.to(torch.int32 if W == 32 else torch.int64), off, lists


class OracleCodec:
    """The calls exchange.PackedExchange makes, on CPU tensors, answered by the oracle."""

    def __init__(self, oracle):
        self.o = oracle

    def compress_bound(self, n, W):
        return self.o.compress_bound(n, W)

    def batch_compress_bound(self, counts, W):
        return self.o.batch_bound(np.concatenate([[0], np.cumsum(counts)]).astype(np.uint64), W)

    def workspace_bytes(self, n, n_buf, W):
        return 16

    def compress_batch_codec(self, rule, ids, in_off, n_buf, W, thr, out, out_off, ws, status):
        a = ids.numpy().view(np.uint32 if W == 32 else np.uint64)
        b, off = self.o.compress_batch(a, in_off.numpy().astype(np.uint64), thr, codec=rule)
        out[:len(b)] = torch.from_numpy(b.copy())
        out_off.copy_(torch.from_numpy(off.astype(np.int64)))

    def decompress_batch(self, d_in, in_off, n_buf, W, ids_out, id_off, ws, status):
        ids, ioff = self.o.decompress_batch(d_in.numpy(), in_off.numpy().astype(np.uint64), W, ids_out.numel())
        ids_out[:len(ids)] = torch.from_numpy(ids.view(np.int32 if W == 32 else np.int64).copy())
        id_off.copy_(torch.from_numpy(ioff.astype(np.int64)))


def _resident(ids, capacity, dev):
    """The rank's frontier array: a fixed allocation (a level that found nothing still has a valid ID pointer)."""
    t = torch.zeros(capacity, dtype=ids.dtype, device=dev)
    t[:ids.numel()] = ids.to(dev)
    return t


def _check_received(rank, P, level, W, ids_out, id_off, dense=False):
    id_off = id_off.cpu()
    for s in range(P):
        want = level_buffers(level, s, P, W, dense=dense)[2][rank]
        got = ids_out[int(id_off[s]):int(id_off[s + 1])].cpu().to(torch.int64)
        assert torch.equal(got, want), f"level {level}: rank {rank} from {s}: {len(got)} IDs, expected {len(want)}"


def _gloo_worker(rank, world, port, W, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    from paper_1704_00513_b200 import exchange
    oracle.build()
    ex = exchange.PackedExchange(OracleCodec(oracle), W, world, 3000, torch.device("cpu"), raw_threshold_bytes=64)
    wire = []
    for level in range(3):
        ids, off, _ = level_buffers(level, rank, world, W)
        ids_out = torch.full((world * 3000,), -1, dtype=ids.dtype)
        id_off = torch.zeros(world + 1, dtype=torch.int64)
        n_send, n_recv = ex.exchange(ids, off, ids_out, id_off)
        _check_received(rank, world, level, W, ids_out, id_off)
        wire.append((n_send, n_recv))
    out[rank] = wire
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("W", [32, 64])
def test_packed_exchange_gloo_world2(W):
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_gloo_worker, args=(2, 29621 + W // 32, W, out), nprocs=2, join=True)
        a, b = out[0], out[1]
        # bytes on the wire add up: what both ranks sent = what both received, level by level
        assert [x[0] + y[0] for x, y in zip(a, b)] == [x[1] + y[1] for x, y in zip(a, b)]


def test_slot_addresses():
    from paper_1704_00513_b200 import exchange
    ptrs = [0x7000_0000_0000, 0x7100_0000_0000, 0x7200_0000_0000]
    got = exchange.slot_addresses(ptrs, rank=2, pitch=4096, parity=1)
    assert got == [p + (3 + 2) * 4096 for p in ptrs]                       # slot set 1 starts behind the P slots of set 0
    # no two (source, parity) pairs share a slot of a destination, and all stay inside 2 P pitch bytes
    seen = set()
    for r in range(3):
        for par in (0, 1):
            for d, a in enumerate(exchange.slot_addresses(ptrs, r, 4096, par)):
                assert (d, a) not in seen and 0 <= a - ptrs[d] <= (2 * 3 - 1) * 4096 and a % 16 == 0
                seen.add((d, a))


# ------------------------------------------------------------------ GPU ------------------------------------------------
@pytest.fixture(scope="module")
def B():
    from paper_1704_00513_b200 import build, binding
    build.build()
    assert torch.cuda.is_available()
    binding.lib()
    return binding


class _LocalSlots:                       # the receive buffers of P ranks on one device: peer memory without peers
    def __init__(self, local, peer_ptrs):
        self.local, self.peer_ptrs = local, peer_ptrs

    def barrier(self):
        pass                             # (one stream: every send is enqueued before any receive)


@pytest.mark.gpu
@pytest.mark.parametrize("W", [32, 64])
def test_slot_exchange_four_ranks_on_one_device(B, oracle_mod, W):
    from paper_1704_00513_b200 import exchange
    dev = torch.device("cuda")
    P, max_ids = 4, 40000
    nbytes = exchange.SlotExchange.receive_bytes(P, max_ids, W, B)
    recv = [torch.full((nbytes,), 0xCD, dtype=torch.uint8, device=dev) for _ in range(P)]
    ptrs = [t.data_ptr() for t in recv]
    ex = [exchange.SlotExchange(B, W, r, P, max_ids, _LocalSlots(recv[r], ptrs), raw_threshold_bytes=64) for r in range(P)]
    for level in range(3):               # slot sets 0, 1, 0
        dense = level == 1
        inputs = [level_buffers(level, r, P, W, dense=dense) for r in range(P)]
        for r in range(P):
            ex[r].send(_resident(inputs[r][0], P * max_ids, dev), inputs[r][1].to(dev))
        outs = []
        for r in range(P):
            ids_out = torch.full((P * max_ids,), -1, dtype=inputs[r][0].dtype, device=dev)
            id_off = torch.zeros(P + 1, dtype=torch.int64, device=dev)
            ex[r].receive(ids_out, id_off)
            outs.append((ids_out, id_off))
        torch.cuda.synchronize()
        for r in range(P):
            assert int(ex[r].status.item()) == 0
            _check_received(r, P, level, W, *outs[r], dense=dense)
        # on the wire: slot s of rank d's current set holds the oracle's stream of what s found for d, and
        # sent_bytes says so
        par = level & 1
        for d in range(P):
            for s in range(P):
                want = oracle_mod.compress(inputs[s][2][d].numpy().astype(np.uint32 if W == 32 else np.uint64), 64)
                base = (par * P + s) * ex[d].pitch
                assert np.array_equal(recv[d][base:base + len(want)].cpu().numpy(), want), f"level {level}: {s} -> {d}"
                assert int(ex[s].sent_bytes[d]) == len(want)


@pytest.mark.gpu
def test_slot_exchange_receive_to_frontier(B):
    """The receive side fused with the frontier update: each rank ORs what it received into the bitmaps of its own vertex
    range, filtered by its visited set. Expected bitmaps from set arithmetic on the lists the sources held."""
    from paper_1704_00513_b200 import exchange
    dev = torch.device("cuda")
    W, P, max_ids, n_vertices = 32, 4, 40000, 1 << 22
    chunk = n_vertices // P
    nbytes = exchange.SlotExchange.receive_bytes(P, max_ids, W, B)
    recv = [torch.zeros(nbytes, dtype=torch.uint8, device=dev) for _ in range(P)]
    ptrs = [t.data_ptr() for t in recv]
    ex = [exchange.SlotExchange(B, W, r, P, max_ids, _LocalSlots(recv[r], ptrs), raw_threshold_bytes=64) for r in range(P)]
    g = torch.Generator().manual_seed(5)
    visited = [(torch.rand(chunk, generator=g) < 0.3) for _ in range(P)]                  # per rank: its own vertices
    frontier = [torch.zeros(chunk, dtype=torch.bool) for _ in range(P)]

    def pack(bits):                                                                     # bool[chunk] -> int32 words, bit v % 32 of word v / 32
        w = bits.view(-1, 32).to(torch.int64) << torch.arange(32, dtype=torch.int64)
        return w.sum(1).to(torch.uint32).view(torch.int32).to(dev)

    d_vis = [pack(v) for v in visited]
    d_fr = [pack(f) for f in frontier]
    n_ids = [torch.zeros(1, dtype=torch.int64, device=dev) for _ in range(P)]
    for level in (0, 1):
        inputs = [level_buffers(level, r, P, W, n_vertices, dense=True) for r in range(P)]
        for r in range(P):
            ex[r].send(_resident(inputs[r][0], P * max_ids, dev), inputs[r][1].to(dev))
        for r in range(P):
            ex[r].receive_to_frontier(d_fr[r], d_vis[r], chunk, r * chunk, n_ids[r])
        torch.cuda.synchronize()
        for d in range(P):
            assert int(ex[d].status.item()) == 0
            got = torch.zeros(chunk, dtype=torch.bool)
            for s in range(P):
                got[inputs[s][2][d] - d * chunk] = True
            new = got & ~visited[d]
            frontier[d] |= new
            visited[d] |= new
            assert int(n_ids[d]) == sum(len(inputs[s][2][d]) for s in range(P))
            assert torch.equal(d_fr[d].cpu(), pack(frontier[d]).cpu()), f"level {level}: frontier of rank {d}"
            assert torch.equal(d_vis[d].cpu(), pack(visited[d]).cpu()), f"level {level}: visited set of rank {d}"


@pytest.fixture(scope="module")
def nccl_world1():
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT="29631", RANK="0", WORLD_SIZE="1")
    torch.cuda.set_device(0)
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda:0"))
    yield dist.group.WORLD
    dist.destroy_process_group()


@pytest.mark.gpu
def test_slot_exchange_symmetric_memory_world1(B, nccl_world1):
    """The real transport objects in a 1-rank group: the receive buffer comes from symmetric memory, the destination
    addresses from its rendezvous, the barrier is the device-side one."""
    from paper_1704_00513_b200 import exchange
    dev, W, P, max_ids = torch.device("cuda:0"), 32, 1, 40000
    slots = exchange.SymmetricSlots(exchange.SlotExchange.receive_bytes(P, max_ids, W, B), dev, nccl_world1)
    assert slots.world == 1 and slots.peer_ptrs == [slots.local.data_ptr()]
    ex = exchange.SlotExchange(B, W, 0, P, max_ids, slots)
    for level in range(3):
        ids, off, _ = level_buffers(level, 0, P, W, dense=True)
        ids_out = torch.full((P * max_ids,), -1, dtype=ids.dtype, device=dev)
        id_off = torch.zeros(P + 1, dtype=torch.int64, device=dev)
        ex.exchange(_resident(ids, P * max_ids, dev), off.to(dev), ids_out, id_off)
        torch.cuda.synchronize()
        assert int(ex.status.item()) == 0
        _check_received(0, P, level, W, ids_out, id_off, dense=True)


@pytest.mark.gpu
def test_packed_exchange_nccl_world1(B, nccl_world1):
    from paper_1704_00513_b200 import exchange
    dev, W, P, max_ids = torch.device("cuda:0"), 64, 1, 40000
    ex = exchange.PackedExchange(B, W, P, max_ids, dev, nccl_world1, raw_threshold_bytes=64)
    for level in range(2):
        ids, off, _ = level_buffers(level, 0, P, W, dense=True)
        ids_out = torch.full((P * max_ids,), -1, dtype=ids.dtype, device=dev)
        id_off = torch.zeros(P + 1, dtype=torch.int64, device=dev)
        n_send, n_recv = ex.exchange(_resident(ids, P * max_ids, dev), off.to(dev), ids_out, id_off)
        torch.cuda.synchronize()
        assert int(ex.status.item()) == 0 and n_send == n_recv > 0
        _check_received(0, P, level, W, ids_out, id_off, dense=True)
