"""python -m paper_2110_11658_b200.pipebench -- print the FP32-pipe micro-benchmarks of cuda:0."""
import json

from . import pipe_bench

if __name__ == "__main__":
    print(json.dumps(pipe_bench(0), indent=1))
