"""Helpers for the -m gpu parity tests: build the CUDA context and its oracle twin on the same inputs."""
import numpy as np

import oracle
import pimd_inputs as pi

MASSES = pi.MASSES_AMU


def make_pair(species, positions, box, P, T, dt, gamma, seed, spec):
    """(gpu, ref) on identical inputs.  spec is a pimd_inputs.NetSpec."""
    import paper_2503_23728_b200 as pb

    gpu = pb.PIMD(species, MASSES, positions, box, P, T, dt, gamma, seed, spec)
    ref = oracle.RefPIMD(species, MASSES, positions, box, P, T, dt, gamma, seed, oracle.RefNet.from_spec(spec))
    return gpu, ref


def pair_from_workload(w):
    return make_pair(w.species, w.positions, w.box, w.P, w.T, w.dt, w.gamma, w.seed, w.net)


def gpu_state(gpu):
    q, p, st = gpu.get_state()
    return q.cpu().numpy(), p.cpu().numpy(), st


def spread_beads(gpu, ref, scale=0.03, seed=3):
    """Inject an identical, bead-dependent state into both sides."""
    q, p, st = ref.get_state()
    q = q + scale * np.random.default_rng(seed).standard_normal(q.shape)
    ref.set_state(q, p, st)
    gpu.set_state(q, p, st)
    return q, p


def assert_forces_close(Fg, Fr, rtol, atol, what=""):
    err = np.abs(Fg - Fr)
    bound = rtol * np.abs(Fr) + atol
    worst = (err - bound).max()
    assert worst <= 0, f"{what}: max |dF| = {err.max():.3e} (|F| max {np.abs(Fr).max():.3e}), violates bound by {worst:.3e}"
