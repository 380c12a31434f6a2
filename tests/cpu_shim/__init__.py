"""TEST INFRASTRUCTURE: host execution of the CUDA kernel sources for `-m "not gpu"` checks (README.md)."""
