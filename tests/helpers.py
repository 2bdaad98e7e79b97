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
