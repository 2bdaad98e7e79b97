"""Small helpers shared by the tests (no method arithmetic)."""
import numpy as np
import torch


def np64(t):
    """torch tensor (any float dtype, any device) -> numpy float64 holding the same values."""
    return t.detach().to("cpu", torch.float64).numpy()


def weights_np64(w):
    """synth.make_weights(...) dict -> the oracle's numpy fp64 dicts."""
    g = {k: np64(v) for k, v in w["global"].items()}
    blocks = [{k: np64(v) for k, v in b.items()} for b in w["blocks"]]
    return g, blocks


def rel_l2(a, b):
    """||a - b||_2 / ||b||_2 over the whole tensor, b = oracle."""
    a = np.asarray(a, dtype=np.float64).reshape(-1)
    b = np.asarray(b, dtype=np.float64).reshape(-1)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


BF16_U = 2.0 ** -8          # unit roundoff of one round-to-nearest bf16 store (8 significand bits)


def elem_excess(got, ref, rel, abs_rms):
    """Per-element parity: max over elements of |got - ref| / (rel * |ref| + abs_rms * rms(ref)).  <= 1 means EVERY
    element is within `rel` of the oracle (one output rounding) plus an absolute floor scaled by the tensor's rms
    (accumulation-order error of elements that cancel to near zero).  A whole-tensor rel-L2 cannot see one wrong
    element in 10^5; this can: a wrong element is off by ~rms(ref), hundreds of times the bound."""
    got = np.asarray(got, dtype=np.float64).reshape(-1)
    ref = np.asarray(ref, dtype=np.float64).reshape(-1)
    if ref.size == 0:
        return 0.0
    rms = float(np.sqrt(np.mean(ref * ref)))
    return bound_excess(got, ref, rel * np.abs(ref) + abs_rms * max(rms, 1e-300))


def bound_excess(got, ref, bound):
    """max over elements of |got - ref| / bound (bound: array of per-element bounds)."""
    got, ref, bound = (np.asarray(a, dtype=np.float64).reshape(-1) for a in (got, ref, bound))
    if ref.size == 0:
        return 0.0
    r = np.abs(got - ref) / bound
    i = int(np.argmax(r))
    if r[i] > 1.0:
        print(f"  bound_excess: worst element #{i}: got {got[i]:.6e} ref {ref[i]:.6e} |err| {abs(got[i] - ref[i]):.3e} bound {bound[i]:.3e}")
    return float(r[i])
