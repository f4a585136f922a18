"""The N > 1 plumbing (paper_2402_05283_b200/dist.py) with world_size 2 over gloo on the CPU:
restart partition, max-over-ranks timing, data broadcast, gather of per-restart errors."""
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_restart_partition_is_a_partition():
    from paper_2402_05283_b200 import dist
    for n in (0, 1, 2, 7, 8, 100):
        for world in (1, 2, 3, 8):
            parts = [dist.restarts_of_rank(n, r, world) for r in range(world)]
            flat = [i for p in parts for i in p]
            assert flat == list(range(n))
            assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1


WORKER = textwrap.dedent("""
    import sys
    sys.path.insert(0, %r)
    import torch
    from paper_2402_05283_b200 import dist
    rank, local_rank, world = dist.init("gloo")
    assert world == 2
    # measured data travels from rank 0
    t = torch.full((4, 8, 8), float(rank + 1))
    m = torch.full((4, 8, 8), rank + 1, dtype=torch.uint8)
    dist.broadcast_arrays([t, m])
    assert float(t.sum()) == 4 * 64 and int(m.sum()) == 4 * 64
    # timing: the slowest rank counts
    assert dist.max_over_ranks(1.0 + rank) == 2.0
    assert dist.sum_over_ranks(1.0 + rank) == 3.0
    # restarts: rank r runs restart r; errors gathered and ranked on every rank
    mine = dist.restarts_of_rank(5, rank, world)
    assert mine == ([0, 1, 2] if rank == 0 else [3, 4])
    ranked = dist.gather_restart_errors([0.5 - 0.1 * i for i in mine], mine)
    assert [i for i, _ in ranked] == [4, 3, 2, 1, 0]
    # Step C across ranks: a stand-in for the device bank (same methods as Plan), episodes = constants
    class Bank:
        def __init__(self, n_keep, eps):
            self.n_keep, self.eps = n_keep, list(eps)
        def merge_errors(self):
            E = torch.zeros(self.n_keep, dtype=torch.float64)
            for i, (e, _) in enumerate(self.eps):
                E[i] = e
            return E, torch.tensor([len(self.eps)], dtype=torch.int32)
        def merge_get(self, slot):
            return self.eps[slot][1].clone()
        def merge_begin(self, n_keep):
            self.n_keep, self.eps = n_keep, []
        def merge_offer(self, ep, E):
            self.eps.append((float(E), ep.clone()))
        def merge_finish(self, n_ref):
            return sorted(self.eps, key=lambda t: t[0])
    ep = lambda v: torch.full((2, 4, 4), complex(v, -v), dtype=torch.complex64)
    bank = Bank(3, [(0.30, ep(1.0)), (0.10, ep(2.0)), (0.50, ep(3.0))] if rank == 0 else [(0.20, ep(4.0)), (0.05, ep(5.0))])
    chosen = dist.select_global_best([e for e, _ in bank.eps], 3)
    assert chosen == [(1, 1, 0.05), (0, 1, 0.10), (1, 0, 0.20)]
    res = dist.merge_across_ranks(bank, 3)
    if rank == 0:
        assert [round(e, 2) for e, _ in res] == [0.05, 0.10, 0.20]
        assert [float(t[0, 0, 0].real) for _, t in res] == [5.0, 2.0, 4.0]
        assert all(t.dtype == torch.complex64 and float(t[1, 3, 3].imag) == -float(t[0, 0, 0].real) for _, t in res)
    else:
        assert res is None
    dist.barrier()
    dist.shutdown()
    print("rank", rank, "ok")
""")


def test_two_ranks_over_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    for r, pr in enumerate(procs):
        out, _ = pr.communicate(timeout=240)
        assert pr.returncode == 0, out
        assert f"rank {r} ok" in out
