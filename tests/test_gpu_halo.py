"""Block decomposition over several contexts: the ranks' contexts run inside one process on the one
GPU this box has, faces move by device copies between the stages (no kernel waits on another).  The decomposed run must
reproduce the single-context run BIT FOR BIT (a shared face's interface flux is evaluated by both sides, bit-identically)
and match the oracle of the whole mesh."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import Oracle                                    # noqa: E402
from oracle.parity import relerr                             # noqa: E402
from paper_2006_15698_b200 import DG                         # noqa: E402
from paper_2006_15698_b200 import decomposed as D            # noqa: E402
from paper_2006_15698_b200 import inputs as I                # noqa: E402

G = 1.4
ORC = Oracle("omp")


def rough_field(nx, ny, nz, p, extent, seed=11):
    return I.density_wave(nx, ny, nz, p, extent, vel=(0.5, -0.3, 0.2), noise=5e-2, seed=seed, waves=(1, 2, 1))


@pytest.mark.parametrize("procs", [(2, 1, 1), (1, 2, 1), (1, 1, 2), (2, 2, 2), (3, 1, 2)])
@pytest.mark.parametrize("p", [1, 3, 4])
def test_decomposed_run_equals_the_single_context_run_bit_for_bit(procs, p):
    n, ext = (7, 6, 5), (1.0, 0.9, 0.8)                        # uneven blocks, ragged columns
    q = rough_field(*n, p, ext)
    dt = I.cfl_dt(ORC.max_wavespeed(q, p, G), p, ext, n, 0.1)
    ranks = D.make_in_process(n, p, G, ext, procs)
    variant = ranks[0].dg.kernel_info()["variant"]
    single = DG(*n, p, G, ext, variant=variant)
    D.set_state_in_process(ranks, q)
    single.set_state(q)
    r_dec, r_one = D.gather_in_process(ranks, "residual"), single.residual()
    assert np.array_equal(r_dec, r_one), relerr(r_dec, r_one)
    assert relerr(r_dec, ORC.residual(q, p, G, ext)) < 1e-11
    D.rk_step_in_process(ranks, dt, 3)
    q_dec, q_one = D.gather_in_process(ranks), single.rk_step(dt, 3).get_state()
    assert np.array_equal(q_dec, q_one), relerr(q_dec, q_one)
    assert relerr(q_dec, ORC.rk_step(q, p, G, ext, dt, 3)) < 1e-12
    lam = max(r.max_wavespeed() for r in ranks)
    assert abs(lam - ORC.max_wavespeed(q_dec, p, G)) <= 4e-16 * lam
    for r in ranks:
        r.close()
    single.close()


@pytest.mark.parametrize("procs", [(2, 1, 1), (1, 1, 2), (2, 2, 2), (3, 2, 1)])
@pytest.mark.parametrize("p", [1, 4, 6])
def test_push_mode_equals_the_single_context_run_bit_for_bit(procs, p):
    """dg_set_halo_pair / dg_set_halo_push: the stage kernels store the face traces straight into the neighbour
    contexts' (double-buffered) halo buffers; no export kernel and no copy between the stages."""
    n, ext = (7, 6, 5), (1.0, 0.9, 0.8)
    q = rough_field(*n, p, ext, seed=5)
    dt = I.cfl_dt(ORC.max_wavespeed(q, p, G), p, ext, n, 0.1)
    ranks = D.make_in_process_push(n, p, G, ext, procs)
    single = DG(*n, p, G, ext, variant=ranks[0].dg.kernel_info()["variant"])
    D.set_state_in_process_push(ranks, q)
    single.set_state(q)
    assert np.array_equal(D.gather_in_process(ranks, "residual"), single.residual())
    launches = sum(r.dg.launch_count for r in ranks)
    D.rk_step_in_process_push(ranks, dt, 3)
    assert sum(r.dg.launch_count for r in ranks) - launches == 15 * len(ranks)      # stage kernels only
    assert np.array_equal(D.gather_in_process(ranks, "residual"), single.rk_step(dt, 3).residual())   # odd parity
    q_dec, q_one = D.gather_in_process(ranks), single.get_state()
    assert np.array_equal(q_dec, q_one), relerr(q_dec, q_one)
    assert relerr(q_dec, ORC.rk_step(q, p, G, ext, dt, 3)) < 1e-12
    for r in ranks:
        r.close()
    single.close()


def test_push_mode_between_two_processes():
    """Two processes, one rank each, the neighbour's halo buffers opened through CUDA IPC and written by the stage kernel
    (tests/push_ipc_worker.py).  Both ranks share this box's one GPU; on a multi-GPU node the same code stores over NVLink."""
    import os
    import socket
    import subprocess
    import sys
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    worker = os.path.join(os.path.dirname(os.path.abspath(__file__)), "push_ipc_worker.py")
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, worker], env=env, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True))
    outs = []
    try:
        for pr in procs:
            outs.append(pr.communicate(timeout=240)[0])
    finally:
        for pr in procs:
            if pr.poll() is None:
                pr.kill()
    for rank, (pr, out) in enumerate(zip(procs, outs)):
        assert pr.returncode == 0 and f"OK rank {rank}" in out, out[-3000:]


def test_decomposition_with_walls_and_far_field():
    n, p, ext = (6, 5, 4), 2, (1.0, 1.0, 0.7)
    bc = (D.WALL, D.FARFIELD, D.PERIODIC, D.PERIODIC, D.WALL, D.WALL)
    qinf = I.uniform_state(1, 1, 1, 0, rho=1.05, vel=(0.45, -0.25, 0.15), pres=1.1, gamma=G).reshape(5)
    q = rough_field(*n, p, ext, seed=4)
    dt = I.cfl_dt(ORC.max_wavespeed(q, p, G), p, ext, n, 0.1)
    ranks = D.make_in_process(n, p, G, ext, (2, 2, 2), bc, qinf)
    assert ranks[0].local_bc == (D.WALL, D.HALO, D.HALO, D.HALO, D.WALL, D.HALO)
    D.set_state_in_process(ranks, q)
    assert relerr(D.gather_in_process(ranks, "residual"), ORC.residual_bc(q, p, G, ext, bc, qinf)) < 1e-11
    D.rk_step_in_process(ranks, dt, 2)
    assert relerr(D.gather_in_process(ranks), ORC.rk_step_bc(q, p, G, ext, bc, qinf, dt, 2)) < 1e-12
    for r in ranks:
        r.close()


def test_halo_faces_need_their_buffers_and_refuse_the_device_side_cfl_step():
    from paper_2006_15698_b200 import DGError
    dg = DG(4, 4, 4, 1).set_boundary((D.HALO, D.HALO, 0, 0, 0, 0))
    q = rough_field(4, 4, 4, 1, (1.0,) * 3)
    dg.set_state(q)
    with pytest.raises(DGError):
        dg.rk_stage(1e-3, 0)                                   # dg_set_halo not called
    with pytest.raises(DGError):
        dg.rk_step_cfl(0.1, 1)                                 # the wavespeed would be this context's only
    # with the buffers in place a single stage runs, but five stages back to back (dg_rk_step) are refused: stages
    # 2..5 would read the neighbours' traces of the first stage.  The state is left alone by the refused call.
    for f in (0, 1):
        dg.set_halo(f, torch.zeros(dg.halo_len(f), dtype=torch.float64, device="cuda"))
    with pytest.raises(DGError) as e:
        dg.rk_step(1e-3, 1)
    assert e.value.code == 2 and "dg_rk_stage" in str(e.value)  # DG_EUNSUPPORTED
    assert np.array_equal(dg.get_state(), q)
    dg.close()


@pytest.mark.parametrize("procs", [(1, 1, 1), (2, 1, 2)])
def test_decomposed_cfl_steps_use_the_global_wavespeed_and_the_librarys_dt(procs):
    """dg_cfl_dt + the maximum of dg_max_wavespeed over the blocks against dg_rk_step_cfl of the single context (whose
    dt comes from the wavespeed fused into the last stage: the kernels' own reciprocal / square root, a few ulp from
    the reduction kernel's, so the two runs agree to rounding, not bit for bit) and against the oracle-driven loop."""
    n, p, ext = (6, 5, 4), 3, (1.0, 0.9, 0.8)
    q = rough_field(*n, p, ext, seed=4)
    ranks = D.make_in_process(n, p, G, ext, procs)
    single = DG(*n, p, G, ext, variant=ranks[0].dg.kernel_info()["variant"])
    D.set_state_in_process(ranks, q)
    if len(ranks) == 1:
        t_dec = ranks[0].rk_step_cfl(0.1, 3)                   # DistributedDG's own method (one rank: no exchange)
    else:
        t_dec = D.rk_step_cfl_in_process(ranks, 0.1, 3)
    t_one, _ = single.set_state(q).rk_step_cfl(0.1, 3)
    q_dec = D.gather_in_process(ranks)
    assert abs(t_dec - t_one) <= 1e-13 * t_one
    assert relerr(q_dec, single.get_state()) < 1e-13
    qo, to = q, 0.0
    for _ in range(3):
        dt = I.cfl_dt(ORC.max_wavespeed(qo, p, G), p, ext, n, 0.1)
        qo, to = ORC.rk_step(qo, p, G, ext, dt, 1), to + dt
    assert abs(t_dec - to) <= 1e-13 * to and relerr(q_dec, qo) < 1e-12
    for r in ranks:
        r.close()
    single.close()
