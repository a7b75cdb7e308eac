"""Re-export of the device plumbing used by the GPU tests."""
from paper_2606_12688_b200.harness import CascadeDecode, DeviceBatch, bf16_tensor, bits_of, f64_of  # noqa: F401
