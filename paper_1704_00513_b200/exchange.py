"""The frontier exchange of one BFS level between the ranks of a process group, with the codec on both sides of it
(Algorithm 4 lines 4-13, L1359-1377: compress -> exchange -> decompress; sizes sent
ahead of the data L1790; compression overlapped with communication L1792-1800, L1834 — the thesis's future work).

One process per GPU. Rank r holds its part of the new frontier as P buffers of ascending IDs, buffer d = the vertices
that rank d owns (`in_offsets`, P + 1 element offsets into one ID array — the layout of bfsc_compress_batch). After the
exchange rank r holds P decoded lists: what every source rank found among the vertices r owns.

Two transports, same result:

* `SlotExchange` — the B200 path (NVLink 5 / NVSwitch peer memory). Every rank owns a receive buffer of 2 x P fixed
  slots in symmetric memory; rank r's stream for rank d is written by the ENCODER ITSELF into slot r of rank d's
  buffer (`bfsc_compress_batch_scatter`: one destination address per stream; the bulk stores of `k_enc_tiles` are the
  transfer). No packed send buffer, no size exchange (a stream carries its size in its header, FORMAT.md §1), no host
  round trip, no copy: encode and send are one kernel, so they overlap by construction. One device-side barrier, then
  `bfsc_decompress_batch` over the rank's own slots. Two slot sets alternate with the level's parity, so a fast rank
  may already write level L + 1 while a slow one still decodes level L (a rank passes the barrier of level L + 1 only
  after its own decode of level L: stream order).
* `PackedExchange` — the portable baseline through the collective library (NCCL, or gloo on CPUs): pack
  (`bfsc_compress_batch`), exchange the P sizes (all-to-all of one int64 per peer, L1790), read them back (the
  collective needs host-side counts), all-to-all-v of the bytes, `bfsc_decompress_batch`.

This module is plumbing: addresses, offsets and collectives. Every byte of every stream is produced and consumed by the
kernels behind the C ABI (`codec` = the binding module; there is no CPU fallback — the tests inject their own codec object
to run the host logic of `PackedExchange` on gloo)."""
import torch
import torch.distributed as dist


def slot_pitch(max_ids_per_buffer: int, W: int, codec) -> int:
    """Bytes between two slots: room for the largest stream of `max_ids_per_buffer` IDs, a multiple of 256."""
    return (codec.compress_bound(max_ids_per_buffer, W) + 255) // 256 * 256


def slot_addresses(peer_ptrs, rank: int, pitch: int, parity: int):
    """Destination of rank `rank`'s stream for every peer d: slot `rank` of slot set `parity` in d's receive buffer
    (2 x P slots of `pitch` bytes behind peer_ptrs[d])."""
    P = len(peer_ptrs)
    return [int(peer_ptrs[d]) + (parity * P + rank) * pitch for d in range(P)]


class SymmetricSlots:
    """The receive buffer of `SlotExchange` in NVLink-mapped symmetric memory (torch.distributed._symmetric_memory):
    `.local` = this rank's 2 x P slots, `.peer_ptrs` = the address of every rank's buffer as seen from this GPU,
    `.barrier()` = a device-side barrier of the group on the current stream."""

    def __init__(self, nbytes: int, device, group=None):
        import torch.distributed._symmetric_memory as symm_mem
        group = group if group is not None else dist.group.WORLD
        self.local = symm_mem.empty(nbytes, dtype=torch.uint8, device=device)
        try:
            self._handle = symm_mem.rendezvous(self.local, group=group)
        except TypeError:
            self._handle = symm_mem.rendezvous(self.local, group.group_name)
        self.peer_ptrs = [int(p) for p in self._handle.buffer_ptrs]
        self.rank, self.world = self._handle.rank, self._handle.world_size

    def barrier(self):
        self._handle.barrier()


class SlotExchange:
    """Peer-memory exchange (see the module text). `slots`: an object with `.local` (uint8 tensor, >= 2 P pitch bytes,
    this rank's receive buffer), `.peer_ptrs` (P addresses) and `.barrier()` — `SymmetricSlots`, or any other mapping of
    peer memory (one process driving several GPUs with peer access enabled, IPC handles)."""

    def __init__(self, codec, W: int, rank: int, n_peers: int, max_ids_per_buffer: int, slots, rule: int = 1,
                 raw_threshold_bytes: int = 0):
        self.codec, self.W, self.rank, self.P = codec, W, rank, n_peers
        self.rule, self.thr = rule, raw_threshold_bytes
        self.max_ids = max_ids_per_buffer
        self.pitch = slot_pitch(max_ids_per_buffer, W, codec)
        self.capacity = codec.compress_bound(max_ids_per_buffer, W)
        self.slots = slots
        assert slots.local.numel() >= 2 * n_peers * self.pitch and len(slots.peer_ptrs) == n_peers
        dev = slots.local.device
        self.dst = [torch.tensor(slot_addresses(slots.peer_ptrs, rank, self.pitch, par), dtype=torch.int64, device=dev)
                    for par in (0, 1)]
        self.slot_off = [self.pitch * torch.arange(par * n_peers, (par + 1) * n_peers + 1, dtype=torch.int64, device=dev)
                         for par in (0, 1)]
        self.sent_bytes = torch.zeros(n_peers, dtype=torch.int64, device=dev)
        total = n_peers * max_ids_per_buffer
        self.ws = torch.empty(codec.workspace_bytes(total, n_peers, W), dtype=torch.uint8, device=dev)
        self.status = torch.zeros(1, dtype=torch.int32, device=dev)
        self.level = 0

    @staticmethod
    def receive_bytes(n_peers: int, max_ids_per_buffer: int, W: int, codec) -> int:
        return 2 * n_peers * slot_pitch(max_ids_per_buffer, W, codec)

    def send(self, ids, in_offsets):
        """Encode this level's P buffers straight into the peers' slots (enqueued on the current stream)."""
        self._par = self.level & 1
        self.level += 1
        self.codec.compress_batch_scatter(self.rule, ids, in_offsets, self.P, self.W, self.thr, self.dst[self._par],
                                          self.capacity, self.sent_bytes, self.ws, self.status)

    def receive(self, ids_out, id_offsets):
        """Decode the own slots of the level last sent (after the barrier) into ids_out (capacity >= P
        max_ids_per_buffer) / id_offsets (P + 1 element offsets: the list received from source rank s is
        ids_out[id_offsets[s] : id_offsets[s + 1]])."""
        self.codec.decompress_batch(self.slots.local, self.slot_off[self._par], self.P, self.W, ids_out, id_offsets,
                                    self.ws, self.status)

    def receive_to_frontier(self, frontier, visited, n_bits, id_base, n_ids):
        """Algorithm 4 lines 10-13 on the own slots in ONE call (`bfsc_decompress_batch_to_frontier`): every received
        vertex that `visited` (bitmap of the rank's own vertices id_base .. id_base + n_bits) does not hold yet is set in
        `visited` and in `frontier`; n_ids (device int64[1]) = IDs received. No ID list is ever written."""
        self.codec.decompress_batch_to_frontier(self.slots.local, self.slot_off[self._par], self.P, self.W, id_base,
                                                frontier, visited, n_bits, n_ids, self.ws, self.status)

    def exchange(self, ids, in_offsets, ids_out, id_offsets):
        """One level, enqueued on the current stream, nothing read back. Errors: `self.status` (device)."""
        self.send(ids, in_offsets)
        self.slots.barrier()                 # every rank's streams of this level have landed
        self.receive(ids_out, id_offsets)


class PackedExchange:
    """Collective-library exchange (see the module text): tensors live where the group's backend wants them (CUDA for
    NCCL, CPU for gloo with an injected codec)."""

    def __init__(self, codec, W: int, n_peers: int, max_ids_per_buffer: int, device, group=None, rule: int = 1,
                 raw_threshold_bytes: int = 0):
        self.codec, self.W, self.P, self.group = codec, W, n_peers, group
        self.rule, self.thr = rule, raw_threshold_bytes
        cap = codec.batch_compress_bound([max_ids_per_buffer] * n_peers, W)
        self.packed = torch.empty(cap, dtype=torch.uint8, device=device)
        self.received = torch.empty(cap, dtype=torch.uint8, device=device)
        self.out_off = torch.zeros(n_peers + 1, dtype=torch.int64, device=device)
        self.recv_off = torch.zeros(n_peers + 1, dtype=torch.int64, device=device)
        self.recv_sizes = torch.zeros(n_peers, dtype=torch.int64, device=device)
        self.ws = torch.empty(codec.workspace_bytes(n_peers * max_ids_per_buffer, n_peers, W), dtype=torch.uint8,
                              device=device)
        self.status = torch.zeros(1, dtype=torch.int32, device=device)

    def exchange(self, ids, in_offsets, ids_out, id_offsets):
        self.codec.compress_batch_codec(self.rule, ids, in_offsets, self.P, self.W, self.thr, self.packed, self.out_off,
                                        self.ws, self.status)
        send_sizes = self.out_off[1:] - self.out_off[:-1]
        dist.all_to_all_single(self.recv_sizes, send_sizes, group=self.group)             # sizes ahead of the data (L1790)
        send_h, recv_h = send_sizes.tolist(), self.recv_sizes.tolist()                    # (the collective needs host counts)
        n_send, n_recv = sum(send_h), sum(recv_h)
        dist.all_to_all_single(self.received[:n_recv], self.packed[:n_send], output_split_sizes=recv_h,
                               input_split_sizes=send_h, group=self.group)
        self.recv_off[1:] = torch.cumsum(self.recv_sizes, 0)
        self.codec.decompress_batch(self.received, self.recv_off, self.P, self.W, ids_out, id_offsets, self.ws,
                                    self.status)
        return n_send, n_recv
