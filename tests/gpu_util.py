"""Re-export of the device plumbing used by the GPU tests."""
from paper_2606_12688_b200.harness import (  # noqa: F401
    DeviceBatch, DeviceBatchFp8, bf16_tensor, bits_of, f64_of)
