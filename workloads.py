"""Seeded synthetic inputs and the BASELINE.json configurations (shapes, sizes, value distributions only).

This module holds none of the method's arithmetic; it serves the tests, bench.py and the oracle-side harness alike.
The tensors stand in for the paper's MNIST / CIFAR-10 / ImageNet workloads: same shapes, seeded
random values with the distributions BASELINE.json states.  Recipe in DESIGN.md section 5."""
import numpy as np

# CKKS parameter sets: kwargs of both paper_2606_16359_b200.Context and (positionally) oracle.ckks.Params
PARAMS = {
    # config 1, primary run: dlen = 1 (beta = 3), reading A1
    "cfg1": dict(log2N=13, n_q=3, q_bits=40, n_p=1, p_bits=60, dnum=3, log2_scale=40),
    # config 1, literal dnum = 1 (dlen = 3): bit-exactness only (P < Q_j, reading A1)
    "cfg1_literal": dict(log2N=13, n_q=3, q_bits=40, n_p=1, p_bits=60, dnum=1, log2_scale=40, allow_noisy_ks=True),
    "cfg2": dict(log2N=14, n_q=8, q_bits=40, n_p=2, p_bits=60, dnum=4, log2_scale=40),
    "cfg3": dict(log2N=16, n_q=24, q_bits=50, n_p=4, p_bits=60, dnum=6, log2_scale=50),
    "cfg4": dict(log2N=16, n_q=30, q_bits=50, n_p=5, p_bits=60, dnum=6, log2_scale=50),
    # small sets for fast parity tests: several tiles, ragged digit (5 limbs, dlen 2 -> digits 2,2,1)
    "toy64": dict(log2N=6, n_q=4, q_bits=30, n_p=2, p_bits=31, dnum=2, log2_scale=25),
    "mid10": dict(log2N=10, n_q=5, q_bits=40, n_p=2, p_bits=60, dnum=3, log2_scale=40),
    "mid12": dict(log2N=12, n_q=5, q_bits=40, n_p=2, p_bits=60, dnum=3, log2_scale=40),
}


def sweep_params(L, dnum):
    """Config 5 (rotation / key-switch sweep), reading A2: dlen = ceil(L/dnum), k = dlen, 50-bit q, 60-bit p."""
    dlen = -(-L // dnum)
    return dict(log2N=16, n_q=L, q_bits=50, n_p=dlen, p_bits=60, dnum=dnum, log2_scale=50)


def oracle_params_args(p):
    """Positional arguments of oracle.ckks.Params for a PARAMS entry."""
    return (p["log2N"], p["n_q"], p["q_bits"], p["n_p"], p["p_bits"], p["dnum"], p["log2_scale"])


# convolution shapes: kwargs of Context.conv_desc / oracle.fragment.ConvDesc
CONVS = {
    "lenet_conv1": dict(BS=1, C_in=1, H=28, W=28, C_out=6, K=5, stride=1, pad=2),          # config 1
    "lenet_conv2": dict(BS=1, C_in=6, H=14, W=14, C_out=16, K=5, stride=1, pad=0),         # config 2 second conv
    "resnet_16_16": dict(BS=1, C_in=16, H=32, W=32, C_out=16, K=3, stride=1, pad=1),       # config 3
    "resnet_16_32_s2": dict(BS=1, C_in=16, H=32, W=32, C_out=32, K=3, stride=2, pad=1),
    "resnet_32_64_s2": dict(BS=1, C_in=32, H=16, W=16, C_out=64, K=3, stride=2, pad=1),
    "fig4_toy": dict(BS=1, C_in=16, H=4, W=4, C_out=16, K=3, stride=1, pad=1),
}


def conv_inputs(seed, conv, x_range=(-1.0, 1.0), w_std=0.1, kaiming=False):
    """x[BS][C_in][H][W] uniform in x_range, w[C_out][C_in or 1][K][K] normal (BASELINE.json configs)."""
    rng = np.random.default_rng(seed)
    x = rng.uniform(x_range[0], x_range[1], (conv["BS"], conv["C_in"], conv["H"], conv["W"]))
    cw = 1 if conv.get("depthwise") else conv["C_in"]
    std = np.sqrt(2.0 / (conv["C_in"] * conv["K"] ** 2)) if kaiming else w_std
    w = rng.normal(0.0, std, (conv["C_out"], cw, conv["K"], conv["K"]))
    return x, w


def random_ct_limbs(seed, q, L, N):
    """uint64 [2][L][N], limb t uniform in [0, q_t) (config 5: "uniform-random limbs mod each prime")."""
    rng = np.random.default_rng(seed)
    out = np.empty((2, L, N), dtype=np.uint64)
    for c in range(2):
        for t in range(L):
            out[c, t] = rng.integers(0, q[t], N, dtype=np.uint64)
    return out


def rotation_steps(seed, count, n):
    """`count` distinct rotation amounts in [1, n-1] (config 5: 32 amounts in [1, 32767])."""
    rng = np.random.default_rng(seed)
    return sorted(int(x) for x in rng.choice(np.arange(1, n), size=count, replace=False))
