"""Small hot-path runs for `compute-sanitizer`: every kernel family once, a few RK4 steps each.

  compute-sanitizer --tool memcheck  python tests/sanitizer_cases.py
  compute-sanitizer --tool racecheck python tests/sanitizer_cases.py
  compute-sanitizer --tool initcheck python tests/sanitizer_cases.py

Not a pytest module (the sanitizer slows kernels down 10-100x; the cases are sized for that).  The summaries of the
last runs are in profiles/r2_sanitizer.md.  Numerics are checked by the parity tests, not here; this script only
prints a checksum per case so that a run that silently did nothing is visible.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import workloads  # noqa: E402
from paper_1803_03498_b200 import Heom  # noqa: E402


def run(name, g, sigma0, dt, steps, full=None):
    if full is not None:
        g.set_full_state(full)
    else:
        g.set_state(sigma0)
    g.rk4_steps(dt, steps)
    k = g.rhs()
    pop, tr = g.populations()
    print(f"{name:34s} kernel={g.kernel_name():26s} nodes={g.nodes:6d} trace={tr.real:+.12f} |rhs|={np.abs(k).max():.6e}")
    g.close()


def main():
    w = workloads.dimer()
    run("dimer, whole-propagation kernel", Heom(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D).bind(),
        w.sigma0(), 1.0, 20)
    run("dimer, stage-wise pipelined", Heom(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D, kernel=2).bind(),
        w.sigma0(), 1.0, 5)
    w = workloads.fmo_like().with_(D=3)
    for form in (-1, 0):
        run(f"7 sites D=3 Hermitian form={form}",
            Heom(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D, rk4_form=form).bind(), w.sigma0(), 1.0, 5)
    g = Heom(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D).bind()
    run("7 sites D=3 general state", g, None, 1.0, 5, full=workloads.random_state(g.nodes, 7, seed=1))
    run("7 sites D=3 generic kernel", Heom(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D, kernel=0).bind(),
        w.sigma0(), 1.0, 3)
    H, bath_state, dip = workloads.with_ground_state(w)
    mu = workloads.dipole_operator(dip, 2).astype(complex)
    s0 = np.zeros_like(mu); s0[:, 0] = mu[:, 0]
    run("absorption, column kernel", Heom(H, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D, bath_state=bath_state).bind(),
        s0, 1.0, 5)
    rng = np.random.default_rng(3)
    H32 = rng.normal(0, 60, (32, 32)); H32 = (H32 + H32.T) / 2
    s0 = np.zeros((32, 32), dtype=complex); s0[0, 0] = 1.0
    run("N=32 D=1 tensor-core, Hermitian", Heom(H32, 35.0, 0.02, 300.0, 0, 1).bind(), s0, 0.5, 3)
    g = Heom(H32, 35.0, 0.02, 300.0, 0, 1).bind()
    run("N=32 D=1 tensor-core, general", g, None, 0.5, 3, full=workloads.random_state(g.nodes, 32, seed=2))
    Hs = rng.normal(0, 60, (7, 7)); Hs = (Hs + Hs.T) / 2
    H29, S, _ = workloads.two_exciton_manifold(Hs)
    s0 = np.zeros((29, 29), dtype=complex); s0[1, 1] = 1.0
    run("two-exciton N=29 D=2, mma kernel", Heom(H29, 35.0, 0.02, 150.0, 0, 2, bath_states=S).bind(), s0, 0.25, 3)
    A = rng.normal(0, 10, (29, 29))
    run("two-exciton N=29 complex H, mma", Heom(H29 + 1j * (A - A.T), 35.0, 0.02, 150.0, 0, 2, bath_states=S).bind(),
        s0, 0.25, 3)
    # one hierarchy as two partitions in one process: pack / unpack kernels of the slice halo
    parts = [Heom(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D, partition=(r, 2)).bind() for r in range(2)]
    import torch
    for g in parts:
        g.set_state(w.sigma0())
        g.rk4_stage(1.0, 0)
        sc, rc = g.partition_plan_slices()[:2]
        per = 2 * g.halo_slice_elements()
        send = torch.zeros(max(1, int(sc.sum())) * per, dtype=torch.float64, device="cuda")
        g.pack_halo_slices(g.stage_output(0), send.data_ptr())
        recv = torch.zeros(max(1, int(rc.sum())) * per, dtype=torch.float64, device="cuda")
        g.unpack_halo_slices(recv.data_ptr(), g.stage_output(0))
        g.sync()
        print(f"partition rank {g.partition[0]}: {int(sc.sum())} pairs packed, {int(rc.sum())} unpacked, checksum {float(send.abs().sum()):.6e}")
        g.close()


if __name__ == "__main__":
    main()
