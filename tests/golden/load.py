"""Reader for tests/golden/paper_values.txt (hand-typed values from the paper)."""
import os


def paper_values():
    out = {}
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "paper_values.txt")
    with open(path) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if not line:
                continue
            key, *vals = line.split()
            nums = [float(v) for v in vals]
            out[key] = nums[0] if len(nums) == 1 else nums
    return out
