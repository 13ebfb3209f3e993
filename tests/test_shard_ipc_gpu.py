"""The fused exchange of the row-sharded path ACROSS PROCESSES: two processes (one rank each) share the one GPU of the
test box, map each other's operand planes through CUDA IPC (mk_ipc_export / mk_ipc_open), attach them
(mk_operand_attach) and run Algorithm 1 with shard.run_row_sharded_fused: the only thing that crosses the process
boundary besides the peer stores of k_fwd / k_post is the host barrier (gloo).  No kernel waits on another process.
Each rank checks its own receiver rows against the fp64 oracle (north_star tolerances) and, bit for bit, against a
single-context run of the same problem."""
import os
import socket

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, regime, q, device_barrier=False):
    import sys
    from pathlib import Path
    sys.path.insert(0, str(Path(__file__).resolve().parent))
    import torch
    import torch.distributed as dist
    from paper_2106_04649_b200 import binding as B, configs, shard
    from _util import gpu_chain, problem, rel_l2
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    torch.cuda.set_device(0)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    opened, mk = [], None
    try:
        cfg = configs.scaled(3, n=45, nt=512, nfoc=19, focal="fan:250", niter=4, A_R=0.02)
        R, Gd, td = problem(cfg)
        whole = gpu_chain(cfg, R, Gd, td, regime=regime, keep_iters=False)
        dev = torch.device("cuda:0")
        rows = shard.row_slice(cfg.n, rank, world)
        mk = B.Marchenko(cfg.n, cfg.n, cfg.nt, cfg.dt, cfg.dx, cfg.fmin, cfg.fmax, rows=(rows.start, len(rows)))
        mk.set_option(B.MK_OPT_EPS_SAMPLES, cfg.eps)
        mk.set_option(B.MK_OPT_REGIME, regime)
        mk.load_R(torch.from_numpy(R).to(dev))
        opened = shard.attach_ipc(mk, cfg.nfoc, dist)

        def host_barrier():
            torch.cuda.synchronize()
            dist.barrier()

        if device_barrier:      # mk_sync_barrier: flag writes / waits on the stream, the host never blocks inside the run
            opened += shard.sync_attach_ipc(mk, dist)
            host_barrier()      # every rank's flags exist and are zero before anyone writes
            barrier = mk.sync_barrier
        else:
            barrier = host_barrier

        names = ("N_last", "f1plus", "f1min", "G", "Gplus", "Gminus")
        outs = {nm: torch.zeros((cfg.nfoc, cfg.n, cfg.nt), dtype=torch.float32, device=dev) for nm in names}
        shard.run_row_sharded_fused(mk, torch.from_numpy(Gd).to(dev), torch.from_numpy(td).to(dev), cfg.niter, outs, barrier)
        host_barrier()
        sl = slice(rows.start, rows.stop)
        worst = max(rel_l2(outs[nm].cpu().numpy()[:, sl], whole[nm][:, sl]) for nm in names)
        alive = float(np.linalg.norm(whole["N_last"])) > 0.0
        # the parity bar proper: this rank's rows against the fp64 oracle (north_star tolerances)
        import oracle
        ref = oracle.marchenko(R, Gd, td, cfg.dt, cfg.dx, cfg.fmin, cfg.fmax, cfg.niter, cfg.eps)
        e_it = rel_l2(outs["N_last"].cpu().numpy()[:, sl], ref["N_iters"][-1][:, sl])
        e_fin = max(rel_l2(outs[nm].cpu().numpy()[:, sl], ref[nm][:, sl]) for nm in names[1:])
        q.put((rank, worst, alive, len(opened) - (world - 1 if device_barrier else 0), e_it, e_fin))
    except Exception as e:   # report instead of hanging the other rank
        q.put((rank, repr(e), False, -1, 1.0, 1.0))
    finally:
        try:
            for p in opened:
                B.ipc_close(p)
            dist.barrier()
        except Exception:
            pass
        if mk is not None:
            mk.close()
        dist.destroy_process_group()


@pytest.mark.parametrize("regime", [2, 3])
def test_two_processes_one_gpu_fused_peer_stores(regime):
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port, world = _free_port(), 2
    procs = [ctx.Process(target=_worker, args=(r, world, port, regime, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=600) for _ in range(world))
    for p in procs:
        p.join(timeout=120)
    print(res)
    for rank, worst, alive, nopened, e_it, e_fin in res:
        assert isinstance(worst, float), worst
        assert alive and worst <= 1e-6
        assert e_it <= 2e-5 and e_fin <= 1e-4, (e_it, e_fin)
        assert nopened == 2                               # one peer x two slots x one plane


@pytest.mark.timeout(300)
def test_two_processes_one_gpu_stream_ordered_barriers():
    """The same run with mk_sync_barrier in place of the host barriers: the flag arrays travel as CUDA
    IPC handles, every barrier of shard.run_row_sharded_fused is two stream memory operations per peer, and the host of
    either process enqueues its whole run without waiting for the other."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port, world = _free_port(), 2
    procs = [ctx.Process(target=_worker, args=(r, world, port, 3, q, True)) for r in range(world)]
    for p in procs:
        p.start()
    try:
        res = sorted(q.get(timeout=240) for _ in range(world))
    finally:
        for p in procs:
            p.join(timeout=30)
            if p.is_alive():
                p.kill()
    print(res)
    for rank, worst, alive, nopened, e_it, e_fin in res:
        assert isinstance(worst, float), worst
        assert alive and worst <= 1e-6
        assert e_it <= 2e-5 and e_fin <= 1e-4, (e_it, e_fin)
