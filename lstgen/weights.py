"""T5-DNN weights: Xavier-uniform from a seed (BASELINE.json configs[0]; PAPER.md:68 gives the
two hidden layers of 32 nodes, the trained weights themselves are not available).

Layout (default network) of the flat fp32 vector handed to both the oracle and the CUDA library
(include/lst.h `dnn_weights`): W1[32][23], b1[32], W2[32][32], b2[32], w3[32], b3  (1857 floats).
Biases are zero (Xavier initialisation).  Generated once here; never regenerated elsewhere.
"""
import numpy as np

N_FEAT = 23
N_HID = 32
N_WEIGHTS = N_HID * N_FEAT + N_HID + N_HID * N_HID + N_HID + N_HID + 1  # 1857


def n_weights(n_feat: int = N_FEAT, n_hidden: int = 2) -> int:
    """W1[32][n_feat], b1[32], (n_hidden - 1) x (W[32][32], b[32]), w_out[32], b_out"""
    return N_HID * n_feat + N_HID + (n_hidden - 1) * (N_HID * N_HID + N_HID) + N_HID + 1


def xavier_weights(seed: int, bias_scale: float = 0.0, n_feat: int = N_FEAT, n_hidden: int = 2) -> np.ndarray:
    """Return the flat weight vector (1857 floats for the default 23 -> 32 -> 32 -> 1). `bias_scale` > 0 draws U(-s, s)
    biases (tests only).  `n_feat` / `n_hidden`: the DNN variants of SPEC.md 4.9 (38 inputs; 1, 3 or 4 hidden layers)."""
    rng = np.random.Generator(np.random.PCG64(int(seed) + 0x5EED))

    def xav(fan_out, fan_in):
        a = np.sqrt(6.0 / (fan_in + fan_out))
        return rng.uniform(-a, a, size=(fan_out, fan_in))

    def bias(n):
        if bias_scale > 0.0:
            return rng.uniform(-bias_scale, bias_scale, size=n)
        return np.zeros(n)

    parts = [xav(N_HID, n_feat).ravel(), bias(N_HID)]
    for _ in range(n_hidden - 1):
        parts += [xav(N_HID, N_HID).ravel(), bias(N_HID)]
    parts += [xav(1, N_HID).ravel(), bias(1)]
    flat = np.concatenate(parts).astype(np.float32)
    assert flat.size == n_weights(n_feat, n_hidden)
    return np.ascontiguousarray(flat)
