"""Writes tests/golden/oracle_tiny.txt from the oracle alone (no CUDA code is imported or run).

The paper prints no worked numeric example of any step of this path, so these values are not the
paper's: they freeze the pinned oracle's results on BASELINE.json configs[0], so that an accidental change to the oracle's
arithmetic shows up as a diff of this file. Regenerate with `python tests/golden/make_golden.py` only together with a
commit message naming the passage or DESIGN.md reading that justifies the change."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import legs_oracle as oracle  # noqa: E402
from paper_2311_18482_b200 import inputs  # noqa: E402  (seeded generators only: no method arithmetic)


def values():
    oracle.build()
    scene = inputs.tiny_scene()
    cam = scene.cameras[0]
    proj = oracle.project(scene, cam, 0)
    tl = oracle.tile_lists(proj, cam)
    fw = oracle.composite_forward(proj, scene.sem, scene.unc, cam)
    up = inputs.upstream_gradient(scene, 0)
    bw = oracle.render_backward(scene, cam, up.reshape(-1, up.shape[2]), mode=0, flags=0)
    di = inputs.decode_inputs(P=64, seed=1)
    f = inputs.bf16_bits_to_f32
    dec = oracle.decode(f(di.feat), [f(w) for w in di.weights], di.biases, f(di.codebook), di.d_clip, f(di.queries))
    idx = np.arange(64) % 128
    ls = oracle.semantic_loss(f(di.feat), np.linspace(0, 1, 64), idx, [f(w) for w in di.weights], di.biases, 1.0, 0.1)
    out = {"D": float(tl["D"]), "vals_checksum": float(tl["vals"].astype(np.int64).sum()),
           "n_contrib_sum": float(fw["n_contrib"].sum())}
    for c in range(14):
        out[f"image_channel_{c}_sum"] = float(fw["out"][:, c].sum())
    for k in ("dmeans", "dscales", "dquats", "dopacities", "dsh", "dsem", "dunc", "dmean2d"):
        out[f"{k}_abs_sum"] = float(np.abs(bw[k]).sum())
    out["decode_probs_entropy_sum"] = float(-(dec["probs"] * np.log(dec["probs"])).sum())
    out["decode_decoded_abs_sum"] = float(np.abs(dec["decoded"]).sum())
    out["decode_rel_sum"] = float(dec["rel"].sum())
    for i, n in enumerate(("L_CE", "L_u", "L_s")):
        out[f"loss_{n}"] = float(ls["loss"][i])
    out["loss_dx_abs_sum"] = float(np.abs(ls["dx"]).sum())
    out["loss_dW1_abs_sum"] = float(np.abs(ls["dW"][1]).sum())
    return out


if __name__ == "__main__":
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_tiny.txt")
    with open(path, "w") as fh:
        fh.write("# written by tests/golden/make_golden.py from oracle/ alone; configs[0] (tiny scene), seed 0\n")
        for k, v in values().items():
            fh.write(f"{k} {v!r}\n")
    print(path)
