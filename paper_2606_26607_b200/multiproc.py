"""One process per GPU: plumbing for the rank-share form of a switch.

Process p of W owns ranks [p*R/W, (p+1)*R/W).  It creates those rank regions in a moebius_arena,
receives the file descriptors of every other rank's physical allocation from the process that owns
it ("exported once ... mapped by its peers"; here POSIX fds over unix sockets instead of
CUDA IPC handles), and maps them at base + r * rank_stride.  A switch is then, in every process:
the same deterministic `moebius_plan`, and for each dependency wave one `moebius_reshard_share`
launch followed by a barrier over `torch.distributed` (gloo or nccl -- it carries no data), then
`moebius_reshard_publish`.  Only marshalling and process plumbing here; all data movement is the
library's kernel storing into / loading from the peers' mapped regions.
"""
from __future__ import annotations

import os
import socket
import time

from . import _binding as B


def owned_ranks(R: int, world: int, rank: int):
    if R % world:
        raise ValueError("R must be divisible by the number of processes")
    per = R // world
    return rank * per, (rank + 1) * per


def _sock_path(sock_dir: str, rank: int) -> str:
    return os.path.join(sock_dir, "moebius_arena_%d.sock" % rank)


def exchange_fds(own: dict, R: int, world: int, rank: int, sock_dir: str, timeout_s: float = 120.0) -> dict:
    """`own` = {rank id: fd} of this process's ranks.  Every process serves its fds on a unix socket
    (SCM_RIGHTS) and fetches the others'.  Returns {rank id: fd} for every rank it does NOT own (the
    caller closes them).  Connections queue in the listen backlog and a thread serves them, so all
    processes can fetch at once without deadlock."""
    import threading
    lo, hi = owned_ranks(R, world, rank)
    assert sorted(own) == list(range(lo, hi))
    srv = socket.socket(socket.AF_UNIX, socket.SOCK_STREAM)
    path = _sock_path(sock_dir, rank)
    if os.path.exists(path):
        os.unlink(path)
    srv.bind(path)
    srv.listen(max(world, 1))
    srv.settimeout(timeout_s)

    def serve():
        for _ in range(world - 1):
            conn, _ = srv.accept()
            socket.send_fds(conn, [b"fds"], [own[r] for r in range(lo, hi)])
            conn.close()

    t = threading.Thread(target=serve, daemon=True)
    t.start()
    got = {}
    for peer in range(world):
        if peer == rank:
            continue
        plo, phi = owned_ranks(R, world, peer)
        deadline = time.time() + timeout_s
        while True:
            c = socket.socket(socket.AF_UNIX, socket.SOCK_STREAM)
            try:
                c.connect(_sock_path(sock_dir, peer))
                break
            except (FileNotFoundError, ConnectionRefusedError):
                c.close()
                if time.time() > deadline:
                    raise TimeoutError("peer %d did not open its socket" % peer)
                time.sleep(0.05)
        c.settimeout(timeout_s)
        _, fds, _, _ = socket.recv_fds(c, 16, phi - plo)
        c.close()
        if len(fds) != phi - plo:
            raise RuntimeError("peer %d sent %d fds, expected %d" % (peer, len(fds), phi - plo))
        got.update(zip(range(plo, phi), fds))
    t.join(timeout_s)
    srv.close()
    os.unlink(path)
    return got


def exchange_arena(arena, R: int, world: int, rank: int, sock_dir: str, timeout_s: float = 120.0):
    """Maps every peer-owned rank region into `arena` (created with this process's own ranks)."""
    lo, hi = owned_ranks(R, world, rank)
    own = {r: B.moebius_arena_export(arena, r) for r in range(lo, hi)}
    try:
        peers = exchange_fds(own, R, world, rank, sock_dir, timeout_s)
    finally:
        for fd in own.values():
            os.close(fd)
    for r, fd in sorted(peers.items()):
        B.moebius_arena_import(arena, r, fd)
        os.close(fd)
    if not B.moebius_arena_ready(arena):
        raise RuntimeError("arena is not fully mapped after the exchange")


def switch(ctx, plan, R: int, world: int, rank: int, barrier, stream_handle: int = 0, sync=None):
    """One switch in this process: its share of every wave, a barrier across processes after each
    (`barrier()` carries no data; `sync()` makes this process's launch complete first), publish."""
    lo, hi = owned_ranks(R, world, rank)
    for wave in range(B.moebius_plan_waves(plan)):
        B.moebius_reshard_share(ctx, plan, lo, hi, wave, stream_handle)
        if sync is not None:
            sync()
        barrier()
    B.moebius_reshard_publish(ctx, plan, stream_handle)
    if sync is not None:
        sync()
    barrier()
