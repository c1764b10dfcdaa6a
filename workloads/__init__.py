"""Seeded synthetic owner sets (BASELINE.json configs C1..C5) -- the ONLY module shared by the oracle side and the
CUDA side.  It holds none of the method's arithmetic: it lists parameter shapes and draws input tensors.

What stands in for what: the paper measures on Qwen-style decoder shapes and a 12-layer
GPT-2-vocabulary LM trained on a token stream; neither data nor weights are needed for an
optimizer step, whose cost depends only on shapes and dtypes.  BASELINE.json's five owner sets stand in for the
paper's models, and seeded Gaussian tensors (weights std 0.02; gradients std 1e-3 with a per-row lognormal(0, 0.5)
scale to mimic heavy-tailed row norms) stand in for training tensors.

Generator: numpy Philox, key = (seed, 4 * tensor_id + kind), counter offset = step; fp32 normals, rounded RNE to the
storage dtype by torch.  Both sides consume the stored bytes, so libm differences cannot matter.

A parameter record is the tuple (block_id, ndim, rows, cols, dtype, flags) of oracle.planner / mfsdp_param_t.
"""
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, field

import numpy as np
import torch

BF16, F32 = 0, 1
ROLE_MATRIX, ROLE_TAIL = 0, 1
POLICY_ROLE_GREEDY, POLICY_SCOPE_GREEDY = 0, 1
METRIC_NUMEL, METRIC_NS_FLOPS = 0, 1
NS_BF16, NS_FP32 = 0, 1
KIND_W, KIND_G, KIND_ROWSCALE, KIND_SHAPE = 0, 1, 2, 3

TORCH_DTYPE = {BF16: torch.bfloat16, F32: torch.float32}


@dataclass
class Workload:
    name: str
    params: list                      # [(block_id, ndim, rows, cols, dtype, flags)]
    seed: int
    world: int = 1
    policy: int = POLICY_ROLE_GREEDY
    metric: int = METRIC_NUMEL
    rank: int = 0                     # -1 = heaviest
    steps: int = 1
    precision: int = NS_BF16
    dtype: int = BF16
    row_lognormal: bool = True        # gradients carry a per-row lognormal(0, 0.5) scale
    spectra: dict = field(default_factory=dict)   # tensor_id -> "inv" | "inv2" | "rank8": gradient with that singular spectrum
    muon: dict = field(default_factory=lambda: dict(lr=0.02, weight_decay=0.01, momentum=0.95, nesterov=1,
                                                    ns_steps=5, a=3.4445, b=-4.7750, c=2.0315, eps=1e-7,
                                                    scale_mode=0))
    adamw: dict = field(default_factory=lambda: dict(lr=1e-3, beta1=0.9, beta2=0.95, eps=1e-8, weight_decay=0.01))


def _layers(n_layers, mats, tails, dtype):
    p = []
    for blk in range(n_layers):
        for rows, cols in mats:
            p.append((blk, 2, rows, cols, dtype, 0))
        for n in tails:
            p.append((blk, 1, n, 1, dtype, 0))
    return p


def c1_tiny():
    """C1: 256x256 and 256x1024 fp32 matrices + one 1-D tail of 1024; NS in fp32; plain Gaussian gradients."""
    params = [(0, 2, 256, 256, F32, 0), (0, 2, 256, 1024, F32, 0), (0, 1, 1024, 1, F32, 0)]
    return Workload("c1_tiny", params, seed=0, precision=NS_FP32, dtype=F32, row_lognormal=False)


def c2_gpt2_small():
    """C2: 12 layers x {768x2304, 768x768, 768x3072, 3072x768} bf16, world 1; tails: 6 x 768 + 1 x 3072 per layer."""
    mats = [(768, 2304), (768, 768), (768, 3072), (3072, 768)]
    tails = [768, 768, 768, 768, 768, 3072, 768]
    return Workload("c2_gpt2_small", _layers(12, mats, tails, BF16), seed=1, steps=10)


def c3_ragged(n=512):
    """C3: 512 bf16 matrices, rows and cols independently uniform on {64,128,192,256,384,512}; one block each."""
    vals = (64, 128, 192, 256, 384, 512)
    rng = np.random.Generator(np.random.Philox(key=[2, KIND_SHAPE]))
    draws = rng.integers(0, 6, size=(n, 2))
    params = [(i, 2, vals[int(draws[i, 0])], vals[int(draws[i, 1])], BF16, 0) for i in range(n)]
    return Workload("c3_ragged", params, seed=2, row_lognormal=False)


def c4_llama8b():
    """C4: Llama-3-8B shapes, 32 layers, two RMSNorm tails of 4096 per layer; 8 ranks, NS-flops greedy, rank 0."""
    mats = [(4096, 4096), (1024, 4096), (1024, 4096), (4096, 4096), (14336, 4096), (14336, 4096), (4096, 14336)]
    return Workload("c4_llama8b_rank0of8", _layers(32, mats, [4096, 4096], BF16), seed=3, world=8,
                    metric=METRIC_NS_FLOPS, rank=0)


def c5_llama70b():
    """C5: Llama-3-70B shapes, 80 layers, two RMSNorm tails of 8192 per layer; 64 ranks, NS-flops greedy, heaviest."""
    mats = [(8192, 8192), (1024, 8192), (1024, 8192), (8192, 8192), (28672, 8192), (28672, 8192), (8192, 28672)]
    return Workload("c5_llama70b_heaviestof64", _layers(80, mats, [8192, 8192], BF16), seed=4, world=64,
                    metric=METRIC_NS_FLOPS, rank=-1)


def paper_qwen16l():
    """The paper's own latency workload as far as its text fixes it ("bf16 Qwen-style decoder-transformer
    shapes (hidden 4096, intermediate 16384, 32 heads ...)", 16 layers over shard span 8; Table 1 / 3: "16L / 3.2B",
    MatrixFSDP optimizer step 87 ms on 8 x A100).  3.2 B / 16 layers = 201 M parameters per layer fits six matrices per
    layer -- q, k, v, o 4096 x 4096, up 16384 x 4096, down 4096 x 16384 (SURVEY.md section 6 inference; the paper lists
    no per-layer shapes, no embedding size) -- plus two RMSNorm vectors.  Planner as the paper describes it: ROLE-GREEDY
    on owner-resident numel, 8 ranks, heaviest rank.  Run with the paper's Muon setting (mu 0.5, K 2)."""
    mats = [(4096, 4096)] * 4 + [(16384, 4096), (4096, 16384)]
    return Workload("paper_qwen16l_3.2b_heaviestof8", _layers(16, mats, [4096, 4096], BF16), seed=5, world=8,
                    metric=METRIC_NUMEL, rank=-1)


def small_ragged(seed=7, dtype=BF16, precision=NS_BF16):
    """Parity-test set the oracle finishes in seconds: several tiles, ragged tails, wide / tall / square, odd pitches."""
    shapes = [(320, 200), (200, 320), (130, 130), (64, 520), (520, 64), (384, 384), (72, 1000), (257, 129), (8, 24)]
    params = [(i // 3, 2, r, c, dtype, 0) for i, (r, c) in enumerate(shapes)]
    params += [(0, 1, 1000, 1, dtype, 0), (0, 1, 7, 1, dtype, 0), (2, 1, 4099, 1, dtype, 0)]
    params.sort(key=lambda p: p[0])
    return Workload("small_ragged", params, seed=seed, precision=precision, dtype=dtype)


def medium_ragged(seed=11, dtype=BF16, precision=NS_BF16):
    """Parity-test set for the 256 x 256 CTA-pair tiles: several pair tiles per matrix, ragged edges in both
    dimensions (not multiples of 64 / 128 / 256), wide / tall / square; still seconds for the oracle."""
    shapes = [(600, 904), (904, 520), (768, 768), (513, 1288), (1288, 264), (256, 256), (1000, 392)]
    params = [(i // 3, 2, r, c, dtype, 0) for i, (r, c) in enumerate(shapes)]
    params += [(0, 1, 513, 1, dtype, 0)]
    params.sort(key=lambda p: p[0])
    return Workload("medium_ragged", params, seed=seed, precision=precision, dtype=dtype)


def edge_shapes(seed=13, dtype=BF16, precision=NS_BF16):
    """Degenerate and boundary shapes: scalars, single rows / columns, exact tile multiples and one past them, very
    thin matrices with a long k loop."""
    shapes = [(1, 1), (1, 24), (24, 1), (7, 3), (128, 128), (129, 257), (255, 513), (256, 512), (16, 4096), (4096, 16)]
    params = [(i // 4, 2, r, c, dtype, 0) for i, (r, c) in enumerate(shapes)]
    params += [(0, 1, 1, 1, dtype, 0), (2, 1, 8, 1, dtype, 0)]
    params.sort(key=lambda p: p[0])
    return Workload("edge_shapes", params, seed=seed, precision=precision, dtype=dtype)


def fused_shapes(seed=19, dtype=BF16, precision=NS_BF16):
    """Shapes of the whole-matrix Newton-Schulz class (min(rows, cols) <= 128, padded X <= 128 KB): the largest that
    fit (128 x 512, 512 x 128), both size classes, d not a multiple of 16 / 64, n not a multiple of 64 / 128, tall and
    wide twins, and neighbours just outside the class (129 x 200, 128 x 576) that stay on the tile kernel."""
    shapes = [(128, 512), (512, 128), (64, 512), (512, 64), (100, 300), (300, 100), (128, 128), (16, 16), (127, 129),
              (33, 500), (500, 33), (128, 448), (65, 257), (257, 65), (96, 192), (1, 200), (200, 1), (129, 200),
              (128, 576), (72, 256)]
    params = [(i // 5, 2, r, c, dtype, 0) for i, (r, c) in enumerate(shapes)]
    params += [(0, 1, 129, 1, dtype, 0)]
    params.sort(key=lambda p: p[0])
    return Workload("fused_shapes", params, seed=seed, precision=precision, dtype=dtype, row_lognormal=True)


def fused2_shapes(seed=23, dtype=BF16, precision=NS_BF16):
    """Shapes of the second whole-matrix Newton-Schulz class (128 < min(rows, cols) <= 256, max <= 512; A and P on
    chip, X streamed): the largest (256 x 512, 512 x 256), d = 192 (half-empty second row block), d and n that are
    not multiples of 16 / 64 / 128, tall and wide twins, one APPLY chunk and several, and neighbours just outside the
    class (256 x 520, 129 x 1024); every column count a multiple of 8, so that the weight update runs inside the
    kernels' last epilogue."""
    shapes = [(256, 512), (512, 256), (192, 384), (384, 192), (256, 256), (200, 504), (504, 200), (136, 136),
              (255, 264), (264, 256), (129, 1024), (440, 144), (256, 520), (130, 136), (248, 392)]
    params = [(i // 4, 2, r, c, dtype, 0) for i, (r, c) in enumerate(shapes)]
    params += [(1, 1, 77, 1, dtype, 0)]
    params.sort(key=lambda p: p[0])
    return Workload("fused2_shapes", params, seed=seed, precision=precision, dtype=dtype, row_lognormal=True)


def fused8_shapes(seed=29, dtype=BF16, precision=NS_BF16):
    """Whole-matrix class (min(rows, cols) <= 128, padded X <= 128 KB) with EVERY column count a multiple of 8, so that
    the weight update runs inside that kernel's last epilogue (one odd column count anywhere in a table sends the whole
    table to the separate update pass), and with nothing else aligned: d not a multiple of 16, n not a multiple of 64,
    tall row counts not multiples of 128, both shared-memory size classes (X <= 64 KB and <= 128 KB), tall / wide twins."""
    shapes = [(100, 304), (304, 72), (72, 256), (120, 200), (200, 120), (8, 24), (104, 488), (488, 104), (56, 56),
              (24, 8), (40, 504), (300, 88)]
    params = [(i // 4, 2, r, c, dtype, 0) for i, (r, c) in enumerate(shapes)]
    params += [(1, 1, 77, 1, dtype, 0)]
    params.sort(key=lambda p: p[0])
    return Workload("fused8_shapes", params, seed=seed, precision=precision, dtype=dtype, row_lognormal=True)


def vocab_embedding(seed=17, dtype=BF16, precision=NS_BF16):
    """The paper's convergence model puts the 50,257 x 768 embedding and the untied LM head on Muon:
    a very tall matrix with an odd row count (GRAM k loop of 786 blocks) next to one ordinary matrix."""
    params = [(0, 2, 50257, 768, dtype, 0), (1, 2, 768, 3072, dtype, 0), (1, 1, 768, 1, dtype, 0)]
    return Workload("vocab_embedding", params, seed=seed, precision=precision, dtype=dtype)


CONFIGS = {"paper16l": paper_qwen16l, "c1": c1_tiny, "c2": c2_gpt2_small, "c3": c3_ragged, "c4": c4_llama8b, "c5": c5_llama70b,
           "small": small_ragged, "medium": medium_ragged, "edge": edge_shapes, "fused": fused_shapes, "fused2": fused2_shapes,
           "fused8": fused8_shapes,
           "vocab": vocab_embedding}


def get(name):
    return CONFIGS[name]()


# ---- tensors -----------------------------------------------------------------------------------------------------
def _rng(seed, tensor_id, kind, step):
    return np.random.Generator(np.random.Philox(key=[seed, 4 * tensor_id + kind], counter=[0, 0, 0, step]))


def _normal(seed, tensor_id, kind, step, n):
    return _rng(seed, tensor_id, kind, step).standard_normal(n, dtype=np.float32)


def weight(wl, tensor_id, rows, cols):
    """W ~ N(0, 0.02), fp32 values before storage rounding, shape (rows, cols)."""
    return (np.float32(0.02) * _normal(wl.seed, tensor_id, KIND_W, 0, rows * cols)).reshape(rows, cols)


def gradient(wl, tensor_id, rows, cols, step, is_tail=False):
    """G ~ N(0, 1e-3), times exp(0.5 xi_row) per stored row when the workload says so (never for tails)."""
    if not is_tail and tensor_id in wl.spectra:
        return _spectral_gradient(wl, tensor_id, rows, cols, step, wl.spectra[tensor_id])
    g = (np.float32(1e-3) * _normal(wl.seed, tensor_id, KIND_G, step, rows * cols)).reshape(rows, cols)
    if wl.row_lognormal and not is_tail:
        xi = _normal(wl.seed, tensor_id, KIND_ROWSCALE, step, rows)
        g *= np.exp(np.float32(0.5) * xi)[:, None]
    return g


def _spectral_gradient(wl, tensor_id, rows, cols, step, kind):
    """G = U diag(sigma) V^T with seeded Haar-like orthonormal factors (QR of Gaussian matrices) and a prescribed
    spectrum: "inv" sigma_i = 1/i, "inv2" sigma_i = 1/i^2, "rank8" eight equal singular values and zeros; scaled to the
    Frobenius norm 1e-3 sqrt(rows cols) of the Gaussian sets.  Ill-conditioned inputs of the Newton-Schulz iteration:
    singular values far below the top one are amplified by ~3.44 per step and never reach 1 within K = 5."""
    d = min(rows, cols)
    rng = _rng(wl.seed, tensor_id, KIND_G, step)
    U, _ = np.linalg.qr(rng.standard_normal((rows, d)))
    V, _ = np.linalg.qr(rng.standard_normal((cols, d)))
    i = np.arange(1, d + 1, dtype=np.float64)
    sig = {"inv": 1.0 / i, "inv2": 1.0 / i ** 2, "rank8": (i <= 8).astype(np.float64)}[kind]
    g = (U * sig) @ V.T
    g *= 1e-3 * np.sqrt(rows * cols) / np.linalg.norm(g)
    return g.astype(np.float32)


def illcond_shapes(seed=37, dtype=BF16, precision=NS_BF16):
    """Ill-conditioned gradients for every Newton-Schulz kernel class: 256 x 1024 and 768 x 768 (tile kernels), 100 x 304
    (whole-matrix class), 200 x 504 (second whole-matrix class), each with the spectra 1/i, 1/i^2 and rank 8."""
    shapes = [(256, 1024), (768, 768), (100, 304), (200, 504)]
    params, spectra = [], {}
    for si, (r, c) in enumerate(shapes):
        for kind in ("inv", "inv2", "rank8"):
            spectra[len(params)] = kind
            params.append((si, 2, r, c, dtype, 0))
    return Workload("illcond_shapes", params, seed=seed, precision=precision, dtype=dtype, spectra=spectra)


CONFIGS["illcond"] = illcond_shapes


def _fields(d):
    if isinstance(d, dict):
        return d["role"], d["param_id"], d["rows"], d["cols"], d["elem_off"]
    return d.role, d.param_id, d.rows, d.cols, d.elem_off


def flat_elems(desc):
    end = [0, 0]
    for d in desc:
        role, _, rows, cols, off = _fields(d)
        end[role] = max(end[role], (off + rows * cols + 63) // 64 * 64)
    return end[0], end[1]


def fill_flat(wl, desc, kind, step=0, role=ROLE_MATRIX, dtype=None, pin=False, threads=8):
    """Rank-flat CPU tensor (storage dtype) of `kind` (KIND_W / KIND_G) for all descriptors of `role`;
    gaps between segments are zero."""
    n = flat_elems(desc)[role]
    tdt = TORCH_DTYPE[wl.dtype if dtype is None else dtype]
    out = torch.zeros(max(n, 1), dtype=tdt, pin_memory=pin)[:n]

    def one(d):
        r, pid, rows, cols, off = _fields(d)
        if r != role:
            return
        if kind == KIND_W:
            a = weight(wl, pid, rows, cols)
        else:
            a = gradient(wl, pid, rows, cols, step, is_tail=(role == ROLE_TAIL))
        out[off:off + rows * cols] = torch.from_numpy(a.reshape(-1)).to(tdt)   # RNE to the storage dtype

    with ThreadPoolExecutor(max_workers=threads) as ex:
        list(ex.map(one, list(desc)))
    return out
