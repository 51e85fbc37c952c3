"""python -m paper_1508_07077_b200.alu_peaks -- print the measured ALU pipe rates of cuda:0 as one JSON line
(hpmc_alu_peaks; thread-instructions per SM per clock, Philox in blocks per SM per clock)."""
import json

from .binding import alu_peaks

if __name__ == "__main__":
    import torch
    torch.cuda.set_device(0)
    alu_peaks()                      # warm-up (instruction cache, clocks)
    print(json.dumps(alu_peaks()))
