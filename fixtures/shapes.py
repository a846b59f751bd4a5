"""Workload shapes: synthetic buffers shaped like the paper's BLSTM acoustic models.

Stand-ins for the SWB-300 / SWB-2000 models of PAPER.md:106 (data and trained weights are
not available; only the parameter SHAPES are used).  BASELINE.json configs 2-4 use 1024
cells per direction; the paper-literal model has 1024 cells per layer = 512 per direction
("over 43 million parameters ... about 165MB") and is kept as an extra.

Segment table (reading R11): per layer and direction {W_ih [4H x in], W_hh [4H x H],
b [4H]}; then bottleneck {W [2H x 256], b [256]}; then softmax {W [256 x 32000], b [32000]}.
Layer-0 input is 260 (40 FMLLR + 100 i-vector + 3x40 logmel); later layers
take 2H (both directions concatenated).
"""


def blstm_segments(layers, hidden_per_dir, input_dim=260, bottleneck=256, outputs=32000):
    """List of (name, n_elements) in model order."""
    H = hidden_per_dir
    segs = []
    for layer in range(layers):
        in_dim = input_dim if layer == 0 else 2 * H
        for d in ("fwd", "bwd"):
            segs.append((f"lstm{layer}.{d}.w_ih", 4 * H * in_dim))
            segs.append((f"lstm{layer}.{d}.w_hh", 4 * H * H))
            segs.append((f"lstm{layer}.{d}.b", 4 * H))
    segs.append(("bottleneck.w", 2 * H * bottleneck))
    segs.append(("bottleneck.b", bottleneck))
    segs.append(("softmax.w", bottleneck * outputs))
    segs.append(("softmax.b", outputs))
    return segs


def total(segs):
    return sum(n for _, n in segs)


# BASELINE.json configs (index = position in BASELINE.json "configs")
SWB300_SEGMENTS = blstm_segments(4, 1024)      # cfg 1: 94 797 312 params, 28 segments
SWB2000_SEGMENTS = blstm_segments(6, 1024)     # cfg 2/3: 145 145 344 params, 40 segments
PAPER_LITERAL_SEGMENTS = blstm_segments(6, 512)  # 43 130 368 params ("165MB")

CONFIGS = {
    "tiny": dict(S=2, G=2, seg_len=[1_000_000], grad="f32", dist="normal", steps=10),
    "swb300": dict(S=16, G=4, seg_len=[total(SWB300_SEGMENTS)], grad="f32", dist="normal", steps=20),
    "swb2000": dict(S=16, G=4, seg_len=[total(SWB2000_SEGMENTS)], grad="f32", dist="normal", steps=20),
    "swb2000_ragged_bf16": dict(S=8, G=8, seg_len=[n for _, n in SWB2000_SEGMENTS], grad="bf16",
                                dist="normal", steps=20),
    "paper_literal": dict(S=8, G=8, seg_len=[total(PAPER_LITERAL_SEGMENTS)], grad="f32",
                          dist="normal", steps=20),
}
HYPER = dict(lr=0.1, momentum=0.9, weight_sd=0.05, grad_scale=1e-3)


def sweep_points(max_bytes=96 * 10 ** 9):
    """BASELINE.json config 5: P = 2^10..2^28 (powers of 4), G in {2,4,8}, S in {2,4,8,16},
    S*G*P*4 B <= 96 GB."""
    pts = []
    for e in range(10, 29, 2):
        for G in (2, 4, 8):
            for S in (2, 4, 8, 16):
                P = 1 << e
                if S * G * P * 4 <= max_bytes:
                    pts.append((P, S, G))
    return pts
