"""T5-DNN weights: Xavier-uniform from a seed (BASELINE.json configs[0]; PAPER.md:68 gives the
two hidden layers of 32 nodes, the trained weights themselves are not available).

Layout of the flat fp32 vector handed to both the oracle and the CUDA library
(include/lst.h `dnn_weights`): W1[32][23], b1[32], W2[32][32], b2[32], w3[32], b3  (1857 floats).
Biases are zero (Xavier initialisation).  Generated once here; never regenerated elsewhere.
"""
import numpy as np

N_FEAT = 23
N_HID = 32
N_WEIGHTS = N_HID * N_FEAT + N_HID + N_HID * N_HID + N_HID + N_HID + 1  # 1857


def xavier_weights(seed: int, bias_scale: float = 0.0) -> np.ndarray:
    """Return the 1857-float weight vector. `bias_scale` > 0 draws U(-s, s) biases (tests only)."""
    rng = np.random.Generator(np.random.PCG64(int(seed) + 0x5EED))

    def xav(fan_out, fan_in):
        a = np.sqrt(6.0 / (fan_in + fan_out))
        return rng.uniform(-a, a, size=(fan_out, fan_in))

    def bias(n):
        if bias_scale > 0.0:
            return rng.uniform(-bias_scale, bias_scale, size=n)
        return np.zeros(n)

    w1 = xav(N_HID, N_FEAT)
    b1 = bias(N_HID)
    w2 = xav(N_HID, N_HID)
    b2 = bias(N_HID)
    w3 = xav(1, N_HID)
    b3 = bias(1)
    flat = np.concatenate([w1.ravel(), b1, w2.ravel(), b2, w3.ravel(), b3]).astype(np.float32)
    assert flat.size == N_WEIGHTS
    return np.ascontiguousarray(flat)
