"""FP64 CPU oracle written from the paper -- test infrastructure, not the product."""
