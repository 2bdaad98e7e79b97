"""-m gpu test of spot_euler_update_static (include/spot_kernels.h): the Euler update + probe reward with the library's
static __device__ scratch, for callers that cannot call cudaMalloc.  Collected LAST on purpose (the run uses
pytest -x).  The existing path (spot_euler_update with a caller buffer) is the reference: same kernels, fixed reduction
order, no atomics (determinism contract, S9), so the outputs must agree bit for bit - and in any case within the
tolerances of tests/test_gpu_kernels.py::test_euler_update_and_reward (1e-7 on x, 1e-5 on the rewards, relative L2).
Two calls in a row, the second SMALLER than the first, so that the array still holds the first call's partial sums beyond
the slots the second call owns: nothing stale may leak into its rewards.
"""
import pytest
import torch

import paper_2606_19004_b200 as spot
from paper_2606_19004_b200 import binding
from synth import hash_normal
from tests.gpu_common import ensure_built
from tests.helpers import np64, rel_l2

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _lib():
    ensure_built()


def _case(seed, B, E):
    x = hash_normal(seed, B * E, 1.0, torch.float32, "cuda").reshape(B, E)
    v = hash_normal(seed + 1, B * E, 1.0, torch.float32, "cuda").reshape(B, E)
    p = hash_normal(seed + 2, E, 1.0, torch.float32, "cuda")
    return x, v, p


def test_static_scratch_euler_update_matches_the_caller_buffer_path_twice_in_a_row():
    cases = [(_case(9100, 16, 1024 * 64), -0.1), (_case(9200, 5, 64 * 64 + 8), -0.125)]     # config-3 latents, then a ragged small one
    refs = [spot.spot_euler_update(x.clone(), v, dt, p) for (x, v, p), dt in cases]
    outs = [(x.clone(), torch.full((x.shape[0],), float("nan"), dtype=torch.float32, device="cuda")) for (x, v, p), dt in cases]
    torch.cuda.synchronize()
    free = []
    for ((x, v, p), dt), (xo, r) in zip(cases, outs):
        free.append(torch.cuda.mem_get_info()[0])
        binding.spot_euler_update_static(xo, v, dt, p, r)
        torch.cuda.synchronize()
    free.append(torch.cuda.mem_get_info()[0])
    for (x_ref, r_ref), (xo, r) in zip(refs, outs):
        assert rel_l2(np64(xo), np64(x_ref)) < 1e-7 and rel_l2(np64(r), np64(r_ref)) < 1e-5
        assert torch.equal(xo, x_ref) and torch.equal(r, r_ref)
    # the second call (the array's address is known by then) takes no device memory
    assert free[2] >= free[1], free


def test_static_scratch_rejects_sizes_beyond_its_maximum_before_any_launch():
    E = 4096 + 4                                               # two partial sums per sequence
    B = binding.STATIC_PARTIALS_MAX // 2 + 1                   # one sequence too many
    x = torch.ones((B, E), dtype=torch.float32, device="cuda")
    v = torch.ones_like(x)
    p = torch.ones(E, dtype=torch.float32, device="cuda")
    r = torch.zeros(B, dtype=torch.float32, device="cuda")
    with pytest.raises(spot.SpotError, match="exceeds the static scratch") as ei:
        binding.spot_euler_update_static(x, v, -1.0, p, r)
    assert ei.value.status_name == "SPOT_ERR_WORKSPACE"
    torch.cuda.synchronize()
    assert bool((x == 1).all()) and not bool(r.any())
    # the largest size that fits (every slot of the array in use) runs and agrees with the caller-buffer path
    x2, v2 = x[:-1].clone(), v[:-1].clone()
    x_ref, r_ref = spot.spot_euler_update(x2.clone(), v2, -0.5, p)
    r2 = torch.empty(B - 1, dtype=torch.float32, device="cuda")
    binding.spot_euler_update_static(x2, v2, -0.5, p, r2)
    assert torch.equal(x2, x_ref) and torch.equal(r2, r_ref)
    assert rel_l2(np64(r2), np64(torch.full_like(r2, 0.5 * E / E ** 0.5))) < 1e-6          # <1, 0.5 * 1> / sqrt(E)
