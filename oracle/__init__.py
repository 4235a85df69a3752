"""CPU oracle -- test infrastructure only (see hough_oracle.c).  Never imported by the product path."""
