"""Worker of tests/test_replicas_gloo.py: launched by torch.distributed.run with world_size 2 on CPU (gloo)."""
import os
import sys
from pathlib import Path

sys.path.insert(0, str(Path(__file__).resolve().parents[1]))

import torch.distributed as dist

from paper_2606_19025_b200 import replicas

dist.init_process_group("gloo")
rank = dist.get_rank()
replicas.barrier()
ms = replicas.max_over_ranks(1.0 + rank)          # rank 1 is the slow one
val = replicas.whole_job_tokens_per_s(1000, ms)
replicas.barrier()
if rank == 0:
    print(f"RESULT world={replicas.world()} ms={ms} value={val}")
dist.destroy_process_group()
