"""Writes the stored expected values under tests/golden/.  Calls ONLY oracle/ and the input generators.

config1_norm.txt: ||K|| of BASELINE.json config 1 (32x32, 128 angles, 4 half-rotations, m = 4 real Fourier table,
lambda2 = 1) from 30 steps of the oracle's power iteration started at rng([0,1,3]) -- SURVEY.md App. A quotes
62.6035 for the same quantity; PAPER.md prints no worked numeric example, so this is a drift guard, not a paper value.
"""
import sys
from pathlib import Path

ROOT = Path(__file__).resolve().parents[2]
sys.path.insert(0, str(ROOT))
from oracle import ref  # noqa: E402
from paper_1809_09725_b200 import synth  # noqa: E402

c = synth.CONFIGS[1]
P = ref.Problem.from_config(c)
L, _ = P.power(synth.rng(1, 3).standard_normal(P.primal_shape), 30)
(Path(__file__).parent / "config1_norm.txt").write_text(f"{L!r}  # ||K||, config 1, oracle power iteration, 30 steps\n")
print(L)
